// net_tc_kernels.cuh -- the per-atom tanh network (rows a2, a6 of DESIGN.md) on the sm_100a tensor cores.
//
// All three network contractions are batched over atoms and run as tcgen05.mma (kind::tf32, fp32 accumulators in
// TMEM) in 3xTF32 (tc05.cuh), which keeps fp32-grade accuracy (parity tolerances of BASELINE.json hold unchanged):
//   k_net_tc<false>  a2: Z = G W0^T -> x = tanh(Z + b0), E_i, C = w1 (1 - x^2) -> E' = s o (C W0), etil
//   k_net_tc<true>   a6: p = (s o D) W0^T -> Hc = w1 d2 p -> h = s o (Hc W0), gbar = e E' + h      (D1.6, C3.8)
//   k_gradw_tc       a6: dL/dW0 = sum_atoms A (x) G + Bc (x) sD, dL/db0 = sum A, dL/dw1 = sum V, dL/db1 = sum e
//                        with A = w1 (e d1 + d2 p), Bc = w1 d1, V = e x + d1 p                    (D1.7-D1.17)
// Atoms are sorted by species; a CTA works on one species and keeps that species' W0 (split hi/lo, in both operand
// arrangements) resident in shared memory while it loops over 128-atom tiles (k_net_tc: two warpgroups, one tile
// each, so that one tile's epilogue overlaps the other's loads and MMAs).
#pragma once
#include "common.cuh"
#include "tc05.cuh"

struct SpeciesMap {
  int start[GNEP_MAX_SPECIES_C + 1];      // sorted-atom range of each species
  int cta_base[GNEP_MAX_SPECIES_C + 1];   // k_net_tc: first (persistent) CTA of each species
  int chunk_base[GNEP_MAX_SPECIES_C + 1]; // k_cgrad_radial: first K-chunk of each species
  int chunk_atoms[GNEP_MAX_SPECIES_C];    // atoms per K-chunk
  int gw_base[GNEP_MAX_SPECIES_C + 1];    // k_gradw_tc: first CTA of each species
  int gw_atoms[GNEP_MAX_SPECIES_C];       // atoms per k_gradw_tc CTA (multiple of GW_KS)
};

__device__ __forceinline__ int species_of_block(const int *base, int T, int b) {
  int t = 0;
  while (t + 1 < T && b >= base[t + 1]) ++t;
  return t;
}

__host__ __device__ inline int pad_to(int x, int m) { return (x + m - 1) / m * m; }

// Layout of the hidden-layer buffers x = tanh(z) and p (written by k_net_tc, read by k_net_tc<true> and k_gradw_tc):
// blocks of 128 atoms (absolute sorted index), inside a block one [128 atoms][16 neurons] panel per chunk of 16 neurons,
//   XT[(a >> 7)][mu >> 4][a & 127][mu & 15],   NnS = Nn padded to 16 neurons per atom.
// A thread-per-atom access of one chunk is then 64 contiguous bytes per lane with consecutive lanes adjacent (a warp
// moves 2 KB of consecutive memory instead of touching 32 rows 4 NnS bytes apart), and a window of 16 consecutive atoms is
// one contiguous kilobyte per chunk for the bulk copies of k_gradw_tc.
__host__ __device__ inline size_t xt_off(int a, int mu, int NnS) {
  return ((size_t)(a >> 7) * (NnS >> 4) + (mu >> 4)) * 2048 + (size_t)(a & 127) * 16 + (mu & 15);
}

// padded problem sizes of the tensor-core kernels
struct NetDims {
  int NnP;   // neurons padded to 16: N of the first contraction, K of the second
  int NdK;   // descriptors padded to 8: K of the first contraction
  int NdN;   // descriptors padded to 16: N of the second contraction
  int abuf;  // floats of one warpgroup's operand buffer
};
__host__ __device__ inline NetDims net_dims(const DevSpec &sp) {
  NetDims d;
  d.NnP = pad_to(sp.Nn, 16); d.NdK = pad_to(sp.Ndes, 8); d.NdN = pad_to(sp.Ndes, 16);
  d.abuf = 128 * (2 * d.NdK > d.NnP ? 2 * d.NdK : d.NnP);
  return d;
}
__host__ __device__ inline size_t net_tc_smem_bytes(const DevSpec &sp, bool bwd) {
  NetDims d = net_dims(sp);
  size_t fl = 2 * (size_t)d.NdK * d.NnP + 2 * (size_t)d.NnP * d.NdN + 2 * d.NnP + d.NdN + 2 * (size_t)d.abuf;
  if (!bwd) fl += 16 * sp.T * sp.KRp;
  return fl * sizeof(float) + 128;
}

// tanh(z) = 1 - 2 / (exp(2 z) + 1) with the hardware exp2 and reciprocal: absolute error <= ~1e-7 over the whole range
// (the argument rounding of exp2 only matters where tanh is already saturated), about 6 instructions.
__device__ __forceinline__ float tanh_fast(float z) {
  float e, rc;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(fminf(z * 2.885390081777927f, 126.f)));   // exp(2 z), no overflow
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rc) : "f"(e + 1.f));
  return fmaf(-2.f, rc, 1.f);
}

// 3xTF32 split with integer round-half-away (2 + 1 + 2 instructions): hi = tf32(x), lo = tf32(x - hi)
__device__ __forceinline__ void split_fast(float x, float &hi, float &lo) {
  hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
  lo = __uint_as_float((__float_as_uint(x - hi) + 0x1000u) & 0xffffe000u);
}
__device__ __forceinline__ void split4_fast(const float4 &x, float4 &hi, float4 &lo) {
  split_fast(x.x, hi.x, lo.x); split_fast(x.y, hi.y, lo.y); split_fast(x.z, hi.z, lo.z); split_fast(x.w, hi.w, lo.w);
}

#define NET_PRE 16      // row chunks (float4) of the next tile held in registers

__device__ __forceinline__ void wg_barrier(int wg) { asm volatile("bar.sync %0, 128;" ::"r"(1 + wg) : "memory"); }

// 4 consecutive values of a row of length W starting at column c (zeros beyond W); vectorised when rows are 16-byte aligned
__device__ __forceinline__ float4 load_row4(const float *__restrict__ row, int W, int c, bool vec, bool valid) {
  float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
  if (!valid) return v;
  if (vec && c + 4 <= W) return *(const float4 *)(row + c);
  if (c < W) v.x = row[c];
  if (c + 1 < W) v.y = row[c + 1];
  if (c + 2 < W) v.z = row[c + 2];
  if (c + 3 < W) v.w = row[c + 3];
  return v;
}
__device__ __forceinline__ void store_row4(float *__restrict__ row, int W, int c, bool vec, float4 v) {
  if (vec && c + 4 <= W) { *(float4 *)(row + c) = v; return; }
  if (c < W) row[c] = v.x;
  if (c + 1 < W) row[c + 1] = v.y;
  if (c + 2 < W) row[c + 2] = v.z;
  if (c + 3 < W) row[c + 3] = v.w;
}

__device__ __forceinline__ void load_row8(const float *__restrict__ row, int W, int c, bool vec4, bool vec8, bool valid, float4 &a, float4 &b) {
  if (valid && vec8 && c + 8 <= W) { const float8 r = ldg256(row + c); a = r.lo; b = r.hi; return; }
  a = load_row4(row, W, c, vec4, valid);
  b = load_row4(row, W, c + 4, vec4, valid);
}
__device__ __forceinline__ void store_row8(float *__restrict__ row, int W, int c, bool vec4, bool vec8, const float4 &a, const float4 &b) {
  if (vec8 && c + 8 <= W) { stg256(row + c, a, b); return; }
  store_row4(row, W, c, vec4, a);
  store_row4(row, W, c + 4, vec4, b);
}

// ------------------------------------------------------------------------------------------------
// a2 / a6: two chained contractions per 128-atom tile.  Thread r of a warpgroup owns atom row r (TMEM lane r).
//   step 1  rows of `in_rows` (q or D), scaled by s, split hi/lo -> K-major operand tile [NdK/4][128][4]
//   step 2  one thread: D1[128][NnP] = rows . W0^T            (3 MMAs per K = 8)
//   step 3  epilogue 1 per (atom, neuron); the second A operand goes back hi -> TMEM (in place of D1), lo -> smem
//   step 4  one thread: D2[128][NdN] = A2 . W0                (A hi from TMEM, lo from smem)
//   step 5  epilogue 2 per (atom, descriptor)
// ------------------------------------------------------------------------------------------------
template <bool BWD>
__global__ void __launch_bounds__(256, 1)
k_net_tc(DevSpec sp, SpeciesMap sm, const float *__restrict__ theta, const float *__restrict__ qscale,
         const float *__restrict__ in_rows, float *__restrict__ xbuf, float *__restrict__ Ei, float *__restrict__ Ep,
         float *__restrict__ etil, const int *__restrict__ struct_s, const float *__restrict__ e_s,
         const float *__restrict__ scales, float *__restrict__ pbuf, float *__restrict__ gbar) {
  using namespace tc05;
  extern __shared__ __align__(128) float smem[];
  const NetDims nd = net_dims(sp);
  const int NnP = nd.NnP, NdK = nd.NdK, NdN = nd.NdN;
  float *W1h = smem, *W1l = W1h + NdK * NnP;             // B of contraction 1: [NdK/4][NnP][4]   (n = mu, k = nu)
  float *W2h = W1l + NdK * NnP, *W2l = W2h + NnP * NdN;  // B of contraction 2: [NnP/4][NdN][4]   (n = nu, k = mu)
  float *b0s = W2l + NnP * NdN, *w1s = b0s + NnP, *qss = w1s + NnP;
  float *cRs = qss + NdN;                                 // forward only: cR[t][J][n][k] as [J*KRp + k][16] (zero padded)
  float *abuf0 = cRs + (BWD ? 0 : 16 * sp.T * sp.KRp);
  uint64_t *bars = (uint64_t *)(abuf0 + 2 * nd.abuf);    // [wg][2]
  uint32_t *tmem_slot = (uint32_t *)(bars + 4);
  const int tid = threadIdx.x, warp = tid >> 5, wg = tid >> 7, r = tid & 127;
  const int t = species_of_block(sm.cta_base, sp.T, blockIdx.x);
  const float *net = theta + sp.offNet + (size_t)t * sp.netSize;

  if (warp == 0) tmem_alloc(tmem_slot, 512);
  if (tid == 32) {
    for (int i = 0; i < 4; ++i) mbar_init(bars + i, 1);
    fence_mbar_init();
  }
  // ---- stage this species' network (zero padded) ----
  for (int x = tid; x < 2 * NdK * NnP + 2 * NnP * NdN; x += 256) smem[x] = 0.f;
  __syncthreads();
  for (int x = tid; x < sp.Nn * sp.Ndes; x += 256) {
    const int mu = x / sp.Ndes, nu = x - mu * sp.Ndes;
    float hi, lo;
    split_tf32(net[x], hi, lo);
    const int o1 = (nu >> 2) * NnP * 4 + mu * 4 + (nu & 3), o2 = (mu >> 2) * NdN * 4 + nu * 4 + (mu & 3);
    W1h[o1] = hi; W1l[o1] = lo; W2h[o2] = hi; W2l[o2] = lo;
  }
  for (int x = tid; x < NnP; x += 256) {
    b0s[x] = x < sp.Nn ? net[sp.Nn * sp.Ndes + x] : 0.f;
    w1s[x] = x < sp.Nn ? net[sp.Nn * sp.Ndes + sp.Nn + x] : 0.f;
  }
  for (int x = tid; x < NdN; x += 256) qss[x] = x < sp.Ndes ? qscale[x] : 0.f;
  if (!BWD)
    for (int x = tid; x < 16 * sp.T * sp.KRp; x += 256) {
      const int o = x >> 4, n = x & 15, J = o / sp.KRp, k = o - J * sp.KRp;
      cRs[x] = (n < sp.NR && k < sp.KR) ? theta[(((size_t)t * sp.T + J) * sp.NR + n) * sp.KR + k] : 0.f;
    }
  fence_async_smem();
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  const uint32_t tbase = *tmem_slot + (uint32_t)(wg * 256);
  // TMEM columns of this warpgroup: D1 main [0,NnP) (later the hi part of the second A operand), D1 corrections
  // [NnP,2NnP); after step 3 the corrections are dead and D2 main / corrections take [NnP,NnP+NdN) / [NnP+NdN,NnP+2NdN).
  // (the accumulator truncates at every accumulation: the small 3xTF32 correction products get their own accumulator)
  const uint32_t tD1 = tbase, tD1c = tbase + NnP, tD2 = tbase + NnP, tD2c = tD2 + NdN;
  const int lane0 = (warp & 3) * 32;
  float *abuf = abuf0 + wg * nd.abuf;
  const uint32_t a1h = smem_u32(abuf), a1l = a1h + (uint32_t)NdK * 128u * 4u;
  const uint32_t w1h_a = smem_u32(W1h), w1l_a = smem_u32(W1l), w2h_a = smem_u32(W2h), w2l_a = smem_u32(W2l);
  const uint32_t id1 = idesc_tf32(128, NnP, 0, 0), id2 = idesc_tf32(128, NdN, 0, 0);
  uint64_t *bar1 = bars + 2 * wg, *bar2 = bar1 + 1;
  const float b1v = net[sp.Nn * sp.Ndes + 2 * sp.Nn];
  const bool vecD = (sp.Ndes & 3) == 0, vecD8 = (sp.Ndes & 7) == 0;
  const int TK = sp.T * sp.KRp;
  const bool vecT = (TK & 3) == 0;

  const int n_t = sm.start[t + 1] - sm.start[t];
  const int tiles = (n_t + 127) >> 7;
  const int ncta = sm.cta_base[t + 1] - sm.cta_base[t];
  uint32_t parity = 0;
  float4 pre[NET_PRE];     // input row of the NEXT tile, requested while the current tile is in its epilogues
  auto prefetch_row = [&](int tile_) {
    const int a_ = sm.start[t] + tile_ * 128 + r;
    const bool ok = tile_ < tiles && a_ < sm.start[t + 1];
    const float *row_ = in_rows + (size_t)a_ * sp.Ndes;
#pragma unroll
    for (int c = 0; c < NET_PRE; c += 2) load_row8(row_, sp.Ndes, 4 * c, vecD, vecD8, ok && c < NdK / 4, pre[c], pre[c + 1]);
  };
  prefetch_row((blockIdx.x - sm.cta_base[t]) * 2 + wg);
  for (int tile = (blockIdx.x - sm.cta_base[t]) * 2 + wg; tile < tiles; tile += 2 * ncta, parity ^= 1u) {
    const int a = sm.start[t] + tile * 128 + r;
    const bool valid = a < sm.start[t + 1];
    // ---- step 1 ---- (the first NET_PRE row chunks were requested during the previous tile)
    {
      const float *row = in_rows + (size_t)a * sp.Ndes;
#pragma unroll
      for (int c = 0; c < NET_PRE; ++c)
        if (c < NdK / 4) {
          float4 v = pre[c];
          const float4 s4 = *(const float4 *)(qss + 4 * c);
          v.x *= s4.x; v.y *= s4.y; v.z *= s4.z; v.w *= s4.w;
          float4 hi, lo;
          split4_fast(v, hi, lo);
          *(float4 *)(abuf + (c * 128 + r) * 4) = hi;
          *(float4 *)(abuf + NdK * 128 + (c * 128 + r) * 4) = lo;
        }
      for (int c = NET_PRE; c < NdK / 4; ++c) {
        float4 v = load_row4(row, sp.Ndes, 4 * c, vecD, valid);
        const float4 s4 = *(const float4 *)(qss + 4 * c);
        v.x *= s4.x; v.y *= s4.y; v.z *= s4.z; v.w *= s4.w;
        float4 hi, lo;
        split4_fast(v, hi, lo);
        *(float4 *)(abuf + (c * 128 + r) * 4) = hi;
        *(float4 *)(abuf + NdK * 128 + (c * 128 + r) * 4) = lo;
      }
    }
    float ev = 0.f;
    if (BWD) {
      ev = valid ? scales[0] * e_s[struct_s[a]] : 0.f;
      if (valid) Ei[a] = ev;   // backward: Ei is the per-atom energy-seed buffer read by k_gradw_tc
    }
    fence_async_smem();
    fence_before_sync();
    wg_barrier(wg);
    // ---- step 2 ----
    if (r == 0) {
      fence_after_sync();
      for (int s = 0; s < NdK / 8; ++s) {
        const uint64_t dah = desc_kmajor(a1h, 128, s), dal = desc_kmajor(a1l, 128, s);
        const uint64_t dbh = desc_kmajor(w1h_a, NnP, s), dbl = desc_kmajor(w1l_a, NnP, s);
        mma_ss(tD1, dah, dbh, id1, s > 0);
        mma_ss(tD1c, dah, dbl, id1, s > 0);
        mma_ss(tD1c, dal, dbh, id1, 1);
      }
      mma_commit(bar1);
    }
    prefetch_row(tile + 2 * ncta);
    float4 xnext[4];   // backward: the x row is fetched one 16-neuron chunk ahead of its use
    if (BWD) {
#pragma unroll
      for (int v = 0; v < 4; v += 2) load_row8(xbuf + xt_off(a, 0, sp.NnS), 16, 4 * v, true, true, valid, xnext[v], xnext[v + 1]);
    }
    if (!mbar_wait(bar1, parity)) __trap();
    fence_after_sync();
    // ---- step 3 ----
    float eacc = 0.f;
    uint32_t tz[16], tc[16];   // TMEM chunk m0 + 16 is in flight while chunk m0 is worked on
    tmem_ld16_issue(tmem_addr(tD1, lane0, 0), tz);
    tmem_ld16_issue(tmem_addr(tD1c, lane0, 0), tc);
    for (int m0 = 0; m0 < NnP; m0 += 16) {
      float z[16], ch[16], cl[16];
      tmem_ld_wait(tz, tc);
#pragma unroll
      for (int i = 0; i < 16; ++i) z[i] = __uint_as_float(tz[i]) + __uint_as_float(tc[i]);
      if (m0 + 16 < NnP) {
        tmem_ld16_issue(tmem_addr(tD1, lane0, m0 + 16), tz);
        tmem_ld16_issue(tmem_addr(tD1c, lane0, m0 + 16), tc);
      }
      if (!BWD) {
        float xs[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const float xv = tanh_fast(z[i] + b0s[m0 + i]);
          const float w1 = w1s[m0 + i];            // zero for padded neurons
          xs[i] = xv;
          eacc += w1 * xv;
          split_fast(w1 * (1.f - xv * xv), ch[i], cl[i]);
        }
        if (valid) {
          float *xr = xbuf + xt_off(a, m0, sp.NnS);
#pragma unroll
          for (int v = 0; v < 2; ++v)
            store_row8(xr, 16, 8 * v, true, true, make_float4(xs[8 * v], xs[8 * v + 1], xs[8 * v + 2], xs[8 * v + 3]),
                       make_float4(xs[8 * v + 4], xs[8 * v + 5], xs[8 * v + 6], xs[8 * v + 7]));
        }
      } else {
        const float *xr = xbuf + xt_off(a, m0 + 16, sp.NnS);   // the next chunk's panel
        float *pr = pbuf + xt_off(a, m0, sp.NnS);
        float4 xcur[4];
#pragma unroll
        for (int v = 0; v < 4; ++v) xcur[v] = xnext[v];
#pragma unroll
        for (int v = 0; v < 4; v += 2) load_row8(xr, 16, 4 * v, true, true, valid && m0 + 16 < NnP, xnext[v], xnext[v + 1]);
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const float4 x4 = xcur[v];
          const float xv[4] = {x4.x, x4.y, x4.z, x4.w};
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float d1 = 1.f - xv[i] * xv[i], d2 = -2.f * xv[i] * d1;
            split_fast(w1s[m0 + 4 * v + i] * d2 * z[4 * v + i], ch[4 * v + i], cl[4 * v + i]);
          }
        }
        if (valid) {
#pragma unroll
          for (int v = 0; v < 2; ++v)
            store_row8(pr, 16, 8 * v, true, true, make_float4(z[8 * v], z[8 * v + 1], z[8 * v + 2], z[8 * v + 3]),
                       make_float4(z[8 * v + 4], z[8 * v + 5], z[8 * v + 6], z[8 * v + 7]));
        }
      }
      {
        float h8[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) h8[i] = ch[i];
        tmem_st8(tmem_addr(tD1, lane0, m0), h8);
#pragma unroll
        for (int i = 0; i < 8; ++i) h8[i] = ch[8 + i];
        tmem_st8(tmem_addr(tD1, lane0, m0 + 8), h8);
      }
#pragma unroll
      for (int v = 0; v < 4; ++v)
        *(float4 *)(abuf + (((m0 >> 2) + v) * 128 + r) * 4) = make_float4(cl[4 * v], cl[4 * v + 1], cl[4 * v + 2], cl[4 * v + 3]);
    }
    if (!BWD && valid) Ei[a] = eacc + b1v;
    tmem_st_wait();
    fence_async_smem();
    fence_before_sync();
    wg_barrier(wg);
    // ---- step 4 ----
    if (r == 0) {
      fence_after_sync();
      for (int s = 0; s < NnP / 8; ++s) {
        const uint64_t dbh = desc_kmajor(w2h_a, NdN, s), dbl = desc_kmajor(w2l_a, NdN, s);
        const uint32_t ta = tmem_addr(tD1, 0, 8 * s);
        mma_ts(tD2, ta, dbh, id2, s > 0);
        mma_ts(tD2c, ta, dbl, id2, s > 0);
        mma_ss(tD2c, desc_kmajor(a1h, 128, s), dbh, id2, 1);
      }
      mma_commit(bar2);
    }
    float4 enext[4];   // backward: E' row, one 16-descriptor chunk ahead
    if (BWD) {
#pragma unroll
      for (int v = 0; v < 4; v += 2) load_row8(Ep + (size_t)a * sp.Ndes, sp.Ndes, 4 * v, vecD, vecD8, valid, enext[v], enext[v + 1]);
    }
    if (!mbar_wait(bar2, parity)) __trap();
    fence_after_sync();
    // ---- step 5 ----
    float epr[16];
    tmem_ld16_issue(tmem_addr(tD2, lane0, 0), tz);
    tmem_ld16_issue(tmem_addr(tD2c, lane0, 0), tc);
    for (int n0 = 0; n0 < NdN; n0 += 16) {
      float v[16];
      tmem_ld_wait(tz, tc);
#pragma unroll
      for (int i = 0; i < 16; ++i) v[i] = (__uint_as_float(tz[i]) + __uint_as_float(tc[i])) * qss[n0 + i];
      if (n0 + 16 < NdN) {
        tmem_ld16_issue(tmem_addr(tD2, lane0, n0 + 16), tz);
        tmem_ld16_issue(tmem_addr(tD2c, lane0, n0 + 16), tc);
      }
      if (!BWD) {
        if (n0 == 0) {
#pragma unroll
          for (int i = 0; i < 16; ++i) epr[i] = v[i];
        }
        if (valid) {
          float *er = Ep + (size_t)a * sp.Ndes;
#pragma unroll
          for (int q8 = 0; q8 < 2; ++q8)
            store_row8(er, sp.Ndes, n0 + 8 * q8, vecD, vecD8, make_float4(v[8 * q8], v[8 * q8 + 1], v[8 * q8 + 2], v[8 * q8 + 3]),
                       make_float4(v[8 * q8 + 4], v[8 * q8 + 5], v[8 * q8 + 6], v[8 * q8 + 7]));
        }
      } else {
        const float *er = Ep + (size_t)a * sp.Ndes;
        float *gr = gbar + (size_t)a * sp.Ndes;
        float4 ecur[4];
#pragma unroll
        for (int q4 = 0; q4 < 4; ++q4) ecur[q4] = enext[q4];
#pragma unroll
        for (int q4 = 0; q4 < 4; q4 += 2) load_row8(er, sp.Ndes, n0 + 16 + 4 * q4, vecD, vecD8, valid && n0 + 16 < NdN, enext[q4], enext[q4 + 1]);
#pragma unroll
        for (int q8 = 0; q8 < 2; ++q8) {
          const float4 ea = ecur[2 * q8], eb = ecur[2 * q8 + 1];
          const int o = 8 * q8;
          if (valid)
            store_row8(gr, sp.Ndes, n0 + o, vecD, vecD8,
                       make_float4(ev * ea.x + v[o], ev * ea.y + v[o + 1], ev * ea.z + v[o + 2], ev * ea.w + v[o + 3]),
                       make_float4(ev * eb.x + v[o + 4], ev * eb.y + v[o + 5], ev * eb.z + v[o + 6], ev * eb.w + v[o + 7]));
        }
      }
    }
    if (!BWD) {   // etil[J][k] = sum_n E'_n cR[t][J][n][k]  (input of the radial force pass)
      float *et = etil + (size_t)a * TK;
      const bool vecT8 = (TK & 7) == 0;
      for (int o = 0; o < TK; o += 8) {
        float acc4[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          if (o + i < TK) {
            const float4 *c4 = (const float4 *)(cRs + (o + i) * 16);
            float s = 0.f;
#pragma unroll
            for (int v = 0; v < 4; ++v) {
              const float4 c = c4[v];
              s += epr[4 * v] * c.x + epr[4 * v + 1] * c.y + epr[4 * v + 2] * c.z + epr[4 * v + 3] * c.w;
            }
            acc4[i] = s;
          }
        }
        if (valid) store_row8(et, TK, o, vecT, vecT8, make_float4(acc4[0], acc4[1], acc4[2], acc4[3]), make_float4(acc4[4], acc4[5], acc4[6], acc4[7]));
      }
    }
    fence_before_sync();   // the next tile's MMAs overwrite D1/D2 and the operand buffer after the barrier of step 1
  }
  fence_before_sync();
  __syncthreads();
  if (warp == 0) tmem_free(*tmem_slot, 512);
}

// ------------------------------------------------------------------------------------------------
// a6: the parameter gradients of the network as ONE contraction over atoms (K = atoms, D1.7-D1.17):
//   D3[mu][nu]   = sum_a A[a][mu] G[a][nu] + Bc[a][mu] sD[a][nu]      (dL/dW0; column nu = Ndes carries G = 1 -> dL/db0)
//   D4[mu][0]    = sum_a V[a][mu]                                       (dL/dw1)
// A, Bc, V are formed on the fly from x, p and the per-atom energy seed e.  Each CTA owns a contiguous atom range of
// one species and walks it in windows of GW_KS atoms aligned to absolute multiples of GW_KS (so that every row block
// is 16-byte aligned for any row length; atoms of a window outside the CTA's range are masked out).
//   warp 9 (one thread)  bulk-copies (cp.async.bulk, mbarrier complete_tx) the raw rows x, p, q, D, e of a window --
//                        five contiguous blocks -- into a ring of `nraw` raw stages;
//   warps 0..7           turn a raw stage into the K-major operand tiles ([atoms/4][row][4], hi/lo split) of one of
//                        GW_OPST operand stages and arrive on its "full" mbarrier;
//   warp 8 (one thread)  issues the MMAs of a full operand stage and commits to its "empty" mbarrier.
// No CTA-wide barrier and no exposed global-load latency sit in the loop.
// The tensor-core accumulator truncates at every accumulation, so the TMEM sums are kept short: a group of
// GW_FLUSH stages accumulates into one of two TMEM sets (hi*hi products and the small 3xTF32 corrections in separate
// accumulators) and is then added, with fp32 rounding, to register accumulators (row mu: threads mu and 128 + mu).
// One partial per CTA is written at the end (reduced in fixed order, fp64, by k_grad_reduce).
// The bulk copies of the last window may read up to GW_KS rows past the end of the arrays: the host pads x, p, q, D, e
// by GW_PAD_ROWS zeroed rows.
// ------------------------------------------------------------------------------------------------
#define GW_KS 16        // atoms per stage (2 MMA K-steps)
#define GW_FLUSH 4      // stages per TMEM accumulation group
#define GW_PROD 256     // producer threads
#define GW_THREADS (GW_PROD + 64)
#define GW_MAXC 4       // 16-column chunks of the accumulator held by one thread (NB <= 112: 7 chunks over two warpgroups)
#define GW_MAXI 4       // work items per producer thread and stage: 4 (Nn + Ndes) <= GW_MAXI * GW_PROD
#define GW_OPST 2       // operand stages
#define GW_MAXRAW 6     // raw stages (at most)
#define GW_PAD_ROWS 32  // zeroed rows the host appends to x, p, q, D, e

__host__ __device__ inline int gw_ncols(const DevSpec &sp) { return pad_to(sp.Ndes + 1, 16); }
__host__ __device__ inline size_t gradw_stage_floats(const DevSpec &sp) {
  return 6 * (size_t)(GW_KS / 4) * 128 * 4 + 4 * (size_t)(GW_KS / 4) * gw_ncols(sp) * 4;
}
__host__ __device__ inline size_t gradw_raw_floats(const DevSpec &sp) { return (size_t)GW_KS * (2 * sp.NnS + 2 * sp.Ndes + 1); }
__host__ __device__ inline size_t gradw_fixed_bytes() { return ((GW_KS / 4) * 16 * 4 + GW_PROD) * sizeof(float) + 256; }
__host__ __device__ inline int gradw_nraw(const DevSpec &sp) {
  const long long left = 227ll * 1024 - (long long)gradw_fixed_bytes() - (long long)(GW_OPST * gradw_stage_floats(sp) * sizeof(float));
  if (left <= 0) return 0;
  const int n = (int)(left / (long long)(gradw_raw_floats(sp) * sizeof(float)));
  return n > GW_MAXRAW ? GW_MAXRAW : n;
}
__host__ __device__ inline size_t gradw_smem_bytes(const DevSpec &sp) {
  return (GW_OPST * gradw_stage_floats(sp) + gradw_nraw(sp) * gradw_raw_floats(sp)) * sizeof(float) + gradw_fixed_bytes();
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(tc05::smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(tc05::smem_u32(bar)), "r"(bytes) : "memory");
}
// contiguous global -> shared bulk copy (16-byte aligned addresses and size), completion counted on an mbarrier
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(tc05::smem_u32(dst)), "l"(__cvta_generic_to_global(src)), "r"(bytes), "r"(tc05::smem_u32(bar))
               : "memory");
}
__global__ void __launch_bounds__(GW_THREADS, 1)
k_gradw_tc(DevSpec sp, SpeciesMap sm, int nraw, const float *__restrict__ theta, const float *__restrict__ qscale,
           const float *__restrict__ eat, const float *__restrict__ q, const float *__restrict__ D,
           const float *__restrict__ x, const float *__restrict__ p, float *__restrict__ partialW,
           float *__restrict__ partialB) {
  using namespace tc05;
  extern __shared__ __align__(128) float smem[];
  constexpr int G4 = GW_KS / 4;                       // atom groups (16-byte K-chunks) per stage
  const int NB = gw_ncols(sp);
  const int tileA = G4 * 128 * 4, tileB = G4 * NB * 4; // floats per operand tile
  const int stage_fl = 6 * tileA + 4 * tileB;
  const int raw_fl = GW_KS * (2 * sp.NnS + 2 * sp.Ndes + 1);
  // operand stage: Ah Al Bh Bl Vh Vl (rows = mu, 128) | Gh Gl Dh Dl (rows = nu, NB);  raw stage: x | p | q | D | e
  float *raw = smem + GW_OPST * stage_fl;
  float *ones = raw + nraw * raw_fl;                  // [G4][16][4]
  float *esh = ones + G4 * 16 * 4;                    // [GW_PROD]
  uint64_t *bars = (uint64_t *)(esh + GW_PROD);
  uint64_t *full = bars, *empty = bars + 2, *group = bars + 4, *rfull = bars + 6, *rempty = bars + 6 + GW_MAXRAW;
  uint32_t *tmem_slot = (uint32_t *)(bars + 6 + 2 * GW_MAXRAW);
  const int tid = threadIdx.x, warp = tid >> 5;
  const int t = species_of_block(sm.gw_base, sp.T, blockIdx.x);
  const float *net = theta + sp.offNet + (size_t)t * sp.netSize;
  const float *w1g = net + sp.Nn * sp.Ndes + sp.Nn;
  const int c0 = sm.start[t] + (blockIdx.x - sm.gw_base[t]) * sm.gw_atoms[t];
  const int c1 = min(c0 + sm.gw_atoms[t], sm.start[t + 1]);
  const int w0 = c0 & ~(GW_KS - 1);                   // first window (absolute multiple of GW_KS)
  if (warp == 0) tmem_alloc(tmem_slot, 512);
  if (tid == 32) {
    for (int i = 0; i < GW_OPST; ++i) { mbar_init(full + i, GW_PROD); mbar_init(empty + i, 1); }
    mbar_init(group, 1); mbar_init(group + 1, 1);
    for (int i = 0; i < GW_MAXRAW; ++i) { mbar_init(rfull + i, 1); mbar_init(rempty + i, GW_PROD); }
    fence_mbar_init();
  }
  for (int i = tid; i < GW_OPST * stage_fl; i += GW_THREADS) smem[i] = 0.f;
  for (int i = tid; i < G4 * 16 * 4; i += GW_THREADS) ones[i] = 1.f;
  __syncthreads();
  // the constant "G = 1" row (nu = Ndes) of every stage's Gh tile
  if (tid < GW_OPST * G4 * 4) {
    const int st = tid / (G4 * 4), rem = tid - st * G4 * 4, g = rem >> 2, i = rem & 3;
    smem[st * stage_fl + 6 * tileA + (g * NB + sp.Ndes) * 4 + i] = 1.f;
  }
  fence_async_smem();
  fence_before_sync();
  __syncthreads();
  fence_after_sync();
  // TMEM set s (two of them): [0,NB) D3 main, [NB,2NB) D3 corrections, [2NB,2NB+16) D4 main, [2NB+16,2NB+32) D4 corr.
  const int setc = 2 * NB + 32;
  const uint32_t tb = *tmem_slot;
  const int nst = (c1 - w0 + GW_KS - 1) / GW_KS;
  const int ngroups = (nst + GW_FLUSH - 1) / GW_FLUSH;

  if (warp == GW_PROD / 32 + 1) {
    // ================= bulk-copy issuer (one thread) =================
    if ((tid & 31) == 0) {
      const uint32_t bx = (uint32_t)(GW_KS * sp.NnS * sizeof(float)), bq = (uint32_t)(GW_KS * sp.Ndes * sizeof(float));
      const uint32_t be = (uint32_t)(GW_KS * sizeof(float)), bx16 = (uint32_t)(GW_KS * 16 * sizeof(float));
      for (int it = 0; it < nst; ++it) {
        const int rs = it % nraw, use = it / nraw;
        if (use > 0 && !mbar_wait(rempty + rs, (uint32_t)((use - 1) & 1))) __trap();
        const size_t a0 = (size_t)(w0 + it * GW_KS);
        float *rb = raw + rs * raw_fl;
        mbar_expect_tx(rfull + rs, 2 * bx + 2 * bq + be);
        for (int c = 0; c < (sp.NnS >> 4); ++c) {     // one contiguous [16 atoms][16 neurons] piece per chunk (XT layout)
          bulk_g2s(rb + c * GW_KS * 16, x + xt_off((int)a0, 16 * c, sp.NnS), bx16, rfull + rs);
          bulk_g2s(rb + GW_KS * sp.NnS + c * GW_KS * 16, p + xt_off((int)a0, 16 * c, sp.NnS), bx16, rfull + rs);
        }
        bulk_g2s(rb + 2 * GW_KS * sp.NnS, q + a0 * sp.Ndes, bq, rfull + rs);
        bulk_g2s(rb + 2 * GW_KS * sp.NnS + GW_KS * sp.Ndes, D + a0 * sp.Ndes, bq, rfull + rs);
        bulk_g2s(rb + 2 * GW_KS * (sp.NnS + sp.Ndes), eat + a0, be, rfull + rs);
      }
    }
  } else if (warp == GW_PROD / 32) {
    // ================= MMA issuer (one thread) =================
    if ((tid & 31) == 0) {
      const uint32_t idW = idesc_tf32(128, NB, 0, 0), id1 = idesc_tf32(128, 16, 0, 0);
      const uint32_t ones_a = smem_u32(ones);
      for (int it = 0; it < nst; ++it) {
        const int st = it % GW_OPST, use = it / GW_OPST, g = it / GW_FLUSH, gi = it - g * GW_FLUSH;
        if (!mbar_wait(full + st, (uint32_t)(use & 1))) __trap();
        fence_after_sync();
        const uint32_t ts = tb + (uint32_t)((g & 1) * setc);
        const uint32_t tM = ts, tC = ts + NB, tV = ts + 2 * NB, tVc = tV + 16;
        const uint32_t sa = smem_u32(smem + st * stage_fl), ga = sa + 6u * (uint32_t)tileA * 4u;
        for (int s = 0; s < GW_KS / 8; ++s) {
          const uint64_t Ah = desc_kmajor(sa, 128, s), Al = desc_kmajor(sa + tileA * 4, 128, s);
          const uint64_t Bh = desc_kmajor(sa + 2 * tileA * 4, 128, s), Bl = desc_kmajor(sa + 3 * tileA * 4, 128, s);
          const uint64_t Vh = desc_kmajor(sa + 4 * tileA * 4, 128, s), Vl = desc_kmajor(sa + 5 * tileA * 4, 128, s);
          const uint64_t Gh = desc_kmajor(ga, NB, s), Gl = desc_kmajor(ga + tileB * 4, NB, s);
          const uint64_t Dh = desc_kmajor(ga + 2 * tileB * 4, NB, s), Dl = desc_kmajor(ga + 3 * tileB * 4, NB, s);
          const uint64_t On = desc_kmajor(ones_a, 16, s);
          const uint32_t acc = (gi > 0 || s > 0) ? 1u : 0u;   // the first K-step of a group overwrites the set
          mma_ss(tM, Ah, Gh, idW, acc);
          mma_ss(tM, Bh, Dh, idW, 1);
          mma_ss(tC, Ah, Gl, idW, acc);
          mma_ss(tC, Al, Gh, idW, 1);
          mma_ss(tC, Bh, Dl, idW, 1);
          mma_ss(tC, Bl, Dh, idW, 1);
          mma_ss(tV, Vh, On, id1, acc);
          mma_ss(tVc, Vl, On, id1, acc);
        }
        mma_commit(empty + st);
        if (gi == GW_FLUSH - 1 || it == nst - 1) mma_commit(group + (g & 1));
      }
    }
  } else {
    // ================= producers (which also hold the register accumulators) =================
    const int nI = G4 * (sp.Nn + sp.Ndes), nA = G4 * sp.Nn;   // work items per stage: (atom group, mu) then (atom group, nu)
    const int lane0 = (warp & 3) * 32;
    float esum = 0.f;
    // Row mu of D3 is held by two threads (TMEM lane mu is visible to warps w and w + 4): thread mu owns the column
    // chunks [0, chalf), thread 128 + mu the chunks [chalf, nch) and D4[mu][0].
    const int wgp = tid >> 7, nch = NB >> 4, chalf = (nch + 1) >> 1, cbeg = wgp ? chalf : 0, ccnt = wgp ? nch - chalf : chalf;
    float racc[GW_MAXC][16], rv = 0.f;
#pragma unroll
    for (int c = 0; c < GW_MAXC; ++c)
#pragma unroll
      for (int i = 0; i < 16; ++i) racc[c][i] = 0.f;
    auto flush = [&](int g) {   // add accumulation group g (complete after its last commit) to the registers
      if (!mbar_wait(group + (g & 1), (uint32_t)((g >> 1) & 1))) __trap();
      fence_after_sync();
      const uint32_t ts = tb + (uint32_t)((g & 1) * setc);
#pragma unroll
      for (int c = 0; c < GW_MAXC; ++c)
        if (c < ccnt) {
          float m[16], k[16];
          tmem_ld16(tmem_addr(ts, lane0, (cbeg + c) * 16), m);
          tmem_ld16(tmem_addr(ts, lane0, NB + (cbeg + c) * 16), k);
#pragma unroll
          for (int i = 0; i < 16; ++i) racc[c][i] += m[i] + k[i];
        }
      if (wgp) {
        float m8[8], k8[8];
        tmem_ld8(tmem_addr(ts, lane0, 2 * NB), m8);
        tmem_ld8(tmem_addr(ts, lane0, 2 * NB + 16), k8);
        rv += m8[0] + k8[0];
      }
      fence_before_sync();
    };
    // The work items of a stage are the same in every stage: (atom group ag, column) of the A-side (x, p -> A, Bc, V)
    // followed by the B-side (q, D -> G, sD).  Each thread decodes its (up to GW_MAXI) items once.
    int r_off[GW_MAXI], s_off[GW_MAXI], i_ag[GW_MAXI], i_kind[GW_MAXI];   // kind: 0 none, 1 A-side, 2 B-side, 3 A-side + sum e
    float i_cf[GW_MAXI];
#pragma unroll
    for (int j = 0; j < GW_MAXI; ++j) {
      const int w = tid + j * GW_PROD;
      i_kind[j] = w < nA ? 1 : (w < nI ? 2 : 0);
      const int wl = w < nA ? w : w - nA, W = w < nA ? sp.Nn : sp.Ndes;
      const int ag = i_kind[j] ? wl / W : 0, col = i_kind[j] ? wl - ag * W : 0;
      i_ag[j] = 4 * ag;
      // raw x / p stage: [neuron chunk][16 atoms][16 neurons]; raw q / D stage: [16 atoms][N_des]
      r_off[j] = i_kind[j] == 1 ? (col >> 4) * GW_KS * 16 + 4 * ag * 16 + (col & 15) : 2 * GW_KS * sp.NnS + 4 * ag * W + col;
      s_off[j] = i_kind[j] == 1 ? (ag * 128 + col) * 4 : 6 * tileA + (ag * NB + col) * 4;
      i_cf[j] = i_kind[j] == 1 ? w1g[col] : (i_kind[j] == 2 ? qscale[col] : 0.f);
      if (i_kind[j] == 1 && col == 0) i_kind[j] = 3;
    }
    const int e_off = 2 * GW_KS * (sp.NnS + sp.Ndes);
    int nfl = 0;                                        // accumulation groups already added to the registers
    int rs = 0, ruse = 0;                               // raw stage of window `it` and how often it has been used: it % nraw,
    for (int it = 0; it < nst; ++it, rs = rs + 1 == nraw ? 0 : rs + 1, ruse += rs == 0) {   // it / nraw without the division
      const int st = it % GW_OPST, use = it / GW_OPST, g = it / GW_FLUSH, gi = it - g * GW_FLUSH;
      float *sb = smem + st * stage_fl;
      const float *rb = raw + rs * raw_fl;
      // group g - 1 is added to the registers one stage late (at the second stage of group g), so that its last
      // MMAs have finished by then; its TMEM set is not written again before group g + 1
      if (gi == (GW_FLUSH > 1 ? 1 : 0) && nfl < g) { flush(nfl); ++nfl; }
      const int a0 = w0 + it * GW_KS;
      const int vlo = c0 - a0, vhi = c1 - a0;         // atoms [vlo, vhi) of the window belong to this CTA
      const bool whole = vlo <= 0 && vhi >= GW_KS;
      if (!mbar_wait(rfull + rs, (uint32_t)(ruse & 1))) __trap();
      if (use > 0 && !mbar_wait(empty + st, (uint32_t)((use - 1) & 1))) __trap();
#pragma unroll
      for (int j = 0; j < GW_MAXI; ++j) {
        if (i_kind[j] == 0) continue;
        float4 hi, lo;
        float *dst = sb + s_off[j];
        const float cf = i_cf[j];
        if (i_kind[j] & 1) {
          const float *rx = rb + r_off[j], *rp = rx + GW_KS * sp.NnS;
          const float4 e4 = *(const float4 *)(rb + e_off + i_ag[j]);
          const float ee[4] = {e4.x, e4.y, e4.z, e4.w};
          float Av[4], Bv[4], Vv[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const bool ok = whole || (i_ag[j] + i >= vlo && i_ag[j] + i < vhi);
            const float xv = rx[i * 16];
            const float pv = ok ? rp[i * 16] : 0.f, ev = ok ? ee[i] : 0.f;
            const float d1 = 1.f - xv * xv, d2 = -2.f * xv * d1;
            Av[i] = cf * (ev * d1 + d2 * pv);
            Bv[i] = ok ? cf * d1 : 0.f;
            Vv[i] = ev * xv + d1 * pv;
            if (i_kind[j] == 3) esum += ev;
          }
          split4_fast(make_float4(Av[0], Av[1], Av[2], Av[3]), hi, lo);
          *(float4 *)(dst) = hi; *(float4 *)(dst + tileA) = lo;
          split4_fast(make_float4(Bv[0], Bv[1], Bv[2], Bv[3]), hi, lo);
          *(float4 *)(dst + 2 * tileA) = hi; *(float4 *)(dst + 3 * tileA) = lo;
          split4_fast(make_float4(Vv[0], Vv[1], Vv[2], Vv[3]), hi, lo);
          *(float4 *)(dst + 4 * tileA) = hi; *(float4 *)(dst + 5 * tileA) = lo;
        } else {
          const float *rq = rb + r_off[j], *rD = rq + GW_KS * sp.Ndes;
          float qv[4], dv[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) { qv[i] = cf * rq[i * sp.Ndes]; dv[i] = cf * rD[i * sp.Ndes]; }
          split4_fast(make_float4(qv[0], qv[1], qv[2], qv[3]), hi, lo);
          *(float4 *)(dst) = hi; *(float4 *)(dst + tileB) = lo;
          split4_fast(make_float4(dv[0], dv[1], dv[2], dv[3]), hi, lo);
          *(float4 *)(dst + 2 * tileB) = hi; *(float4 *)(dst + 3 * tileB) = lo;
        }
      }
      fence_async_smem();
      mbar_arrive(full + st);
      mbar_arrive(rempty + rs);
    }
    for (; nfl < ngroups; ++nfl) flush(nfl);
    esh[tid] = esum;
    // results: row mu lives in threads mu and 128 + mu
    asm volatile("bar.sync 1, %0;" ::"n"(GW_PROD) : "memory");
    const int nb = 2 * sp.Nn + 1;
    float *outW = partialW + (size_t)blockIdx.x * sp.Nn * sp.Ndes;
    float *outB = partialB + (size_t)blockIdx.x * nb;
    if ((tid & 127) < sp.Nn) {
      const int mu = tid & 127;
#pragma unroll
      for (int c = 0; c < GW_MAXC; ++c)
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          const int nu = (cbeg + c) * 16 + i;
          if (c < ccnt) {
            if (nu < sp.Ndes) outW[mu * sp.Ndes + nu] = racc[c][i];
            else if (nu == sp.Ndes) outB[mu] = racc[c][i];
          }
        }
      if (wgp) outB[sp.Nn + mu] = rv;
    }
    if (tid == 0) {
      float s = 0.f;
      for (int i = 0; i < GW_PROD; ++i) s += esh[i];
      outB[2 * sp.Nn] = s;
    }
  }
  fence_before_sync();
  __syncthreads();
  if (warp == 0) tmem_free(tb, 512);
}
