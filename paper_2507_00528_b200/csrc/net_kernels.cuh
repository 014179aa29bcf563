// net_kernels.cuh -- per-atom tanh network (rows a2, a6 of DESIGN.md) and the two "K = atoms" contractions
// that produce the W0 and c^R gradients (rows a6, a7-radial).  Atoms are sorted by species, so every CTA
// works on one species and stages only that species' weights in shared memory.
// Warp tile = GNEP_TILE (8) atoms: one W0 element is loaded once and used for 8 atoms.
#pragma once
#include "common.cuh"

struct SpeciesMap {
  int start[GNEP_MAX_SPECIES_C + 1];      // sorted-atom range of each species
  int cta_base[GNEP_MAX_SPECIES_C + 1];   // first CTA (of GNEP_WARPS*GNEP_TILE atoms) of each species
  int chunk_base[GNEP_MAX_SPECIES_C + 1]; // first K-chunk of each species (gradient contractions)
  int chunk_atoms[GNEP_MAX_SPECIES_C];    // atoms per K-chunk
};

__device__ __forceinline__ int species_of_block(const int *base, int T, int b) {
  int t = 0;
  while (t + 1 < T && b >= base[t + 1]) ++t;
  return t;
}

// shared-memory staging of one species' network: W0 with padded stride ldW, b0, w1, b1, q_scale
struct NetSmem { float *W0, *b0, *w1, *b1, *qs; };
__device__ __forceinline__ float *stage_net(const DevSpec &sp, float *smem, const float *__restrict__ theta,
                                            const float *__restrict__ qscale, int t, NetSmem &ns) {
  ns.W0 = smem;
  ns.b0 = ns.W0 + sp.Nn * sp.ldW;
  ns.w1 = ns.b0 + sp.Nn;
  ns.b1 = ns.w1 + sp.Nn;
  ns.qs = ns.b1 + 1;
  const float *src = theta + sp.offNet + (size_t)t * sp.netSize;
  for (int x = threadIdx.x; x < sp.Nn * sp.Ndes; x += blockDim.x) {
    int mu = x / sp.Ndes, nu = x - mu * sp.Ndes;
    ns.W0[mu * sp.ldW + nu] = src[x];
  }
  for (int x = threadIdx.x; x < 2 * sp.Nn + 1; x += blockDim.x) ns.b0[x] = src[sp.Nn * sp.Ndes + x];
  for (int x = threadIdx.x; x < sp.Ndes; x += blockDim.x) ns.qs[x] = qscale[x];
  int used = sp.Nn * sp.ldW + 2 * sp.Nn + 1 + sp.Ndes;
  return smem + ((used + 3) & ~3);
}
__host__ __device__ inline int net_smem_floats(const DevSpec &sp) {
  return ((sp.Nn * sp.ldW + 2 * sp.Nn + 1 + sp.Ndes) + 3) & ~3;
}


// acc0[a] += w0 * row[a], acc1[a] += w1 * row[a] for the 16 atoms of a warp tile (row: 16 floats in shared memory,
// broadcast LDS.128): 2 outputs x 16 atoms per lane -> 6 shared wavefronts per 32 FMA.
__device__ __forceinline__ void fma16x2(float (&acc0)[GNEP_TILE], float (&acc1)[GNEP_TILE], float w0, float w1,
                                        const float *row) {
#pragma unroll
  for (int v = 0; v < GNEP_TILE / 4; ++v) {
    float4 g = *(const float4 *)(row + 4 * v);
    acc0[4 * v] += w0 * g.x; acc0[4 * v + 1] += w0 * g.y; acc0[4 * v + 2] += w0 * g.z; acc0[4 * v + 3] += w0 * g.w;
    acc1[4 * v] += w1 * g.x; acc1[4 * v + 1] += w1 * g.y; acc1[4 * v + 2] += w1 * g.z; acc1[4 * v + 3] += w1 * g.w;
  }
}

// per-warp tile coordinates: atoms [a0, a0+na) of species t
__device__ __forceinline__ void net_tile(const SpeciesMap &sm, int t, int &a0, int &na) {
  a0 = sm.start[t] + ((blockIdx.x - sm.cta_base[t]) * GNEP_WARPS + (threadIdx.x >> 5)) * GNEP_TILE;
  na = min(GNEP_TILE, sm.start[t + 1] - a0);
}

// stage rows[a0..a0+na) (row length W, optional per-column scale) transposed into dst[col][16] (zeros for a >= na)
__device__ __forceinline__ void stage_rows_t(float *dst, const float *__restrict__ src, const float *scale, int a0, int na,
                                             int W, int lane) {
  for (int a = 0; a < GNEP_TILE; ++a)
    for (int c = lane; c < W; c += 32)
      dst[c * GNEP_TILE + a] = a < na ? (scale ? scale[c] : 1.f) * src[(size_t)(a0 + a) * W + c] : 0.f;
}

// ------------------------------------------------------------------------------------------------
// a2: z = W0 (s o q) + b0, x = tanh z, E_i = w1.x + b1, E'_nu = s_nu sum_mu w1_mu (1-x_mu^2) W0_mu,nu
// (paper Eq.D1.1-D1.5) and etil[J][k] = sum_n E'_n cR[I][J][n][k] for the radial force pass.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_net_fwd(DevSpec sp, SpeciesMap sm, const float *__restrict__ theta, const float *__restrict__ qscale,
          const float *__restrict__ q, float *__restrict__ xout, float *__restrict__ Ei,
          float *__restrict__ Ep, float *__restrict__ etil) {
  extern __shared__ __align__(16) float smem[];
  const int t = species_of_block(sm.cta_base, sp.T, blockIdx.x);
  NetSmem ns;
  float *nxt = stage_net(sp, smem, theta, qscale, t, ns);
  float *cRs = nxt;                                   // cR[t][J][n][k] padded to KRp: [T*NR][KRp]
  const int ncr = (sp.T * sp.NR * sp.KRp + 3) & ~3;
  for (int x = threadIdx.x; x < sp.T * sp.NR * sp.KRp; x += blockDim.x) {
    int row = x / sp.KRp, k = x - row * sp.KRp;
    cRs[x] = k < sp.KR ? theta[((size_t)t * sp.T * sp.NR + row) * sp.KR + k] : 0.f;
  }
  const int per_warp = (sp.Ndes + sp.Nn + sp.NR) * GNEP_TILE;
  float *G = nxt + ncr + (threadIdx.x >> 5) * per_warp;   // [Ndes][16]
  float *Cm = G + sp.Ndes * GNEP_TILE;                     // [Nn][16]
  float *EpR = Cm + sp.Nn * GNEP_TILE;                     // [NR][16]
  __syncthreads();
  const int lane = threadIdx.x & 31;
  int a0, na;
  net_tile(sm, t, a0, na);
  if (na <= 0) return;
  stage_rows_t(G, q, ns.qs, a0, na, sp.Ndes, lane);
  __syncwarp();
  float epart[GNEP_TILE];
#pragma unroll
  for (int a = 0; a < GNEP_TILE; ++a) epart[a] = 0.f;
  for (int m0 = 0; m0 < sp.Nn; m0 += 64) {
    const int mu0 = m0 + lane, mu1 = mu0 + 32;
    const bool ok0 = mu0 < sp.Nn, ok1 = mu1 < sp.Nn;
    const float *w0p = ns.W0 + (ok0 ? mu0 : 0) * sp.ldW, *w1p = ns.W0 + (ok1 ? mu1 : 0) * sp.ldW;
    float acc0[GNEP_TILE], acc1[GNEP_TILE];
    const float b0 = ok0 ? ns.b0[mu0] : 0.f, b1 = ok1 ? ns.b0[mu1] : 0.f;
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) { acc0[a] = b0; acc1[a] = b1; }
    for (int nu = 0; nu < sp.Ndes; ++nu) fma16x2(acc0, acc1, w0p[nu], w1p[nu], G + nu * GNEP_TILE);
    if (ok0) {
      const float w1 = ns.w1[mu0];
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a) {
        float xv = tanhf(acc0[a]);
        if (a < na) xout[(size_t)(a0 + a) * sp.Nn + mu0] = xv;
        Cm[mu0 * GNEP_TILE + a] = w1 * (1.f - xv * xv);
        epart[a] += w1 * xv;
      }
    }
    if (ok1) {
      const float w1 = ns.w1[mu1];
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a) {
        float xv = tanhf(acc1[a]);
        if (a < na) xout[(size_t)(a0 + a) * sp.Nn + mu1] = xv;
        Cm[mu1 * GNEP_TILE + a] = w1 * (1.f - xv * xv);
        epart[a] += w1 * xv;
      }
    }
  }
  __syncwarp();
#pragma unroll
  for (int a = 0; a < GNEP_TILE; ++a) {
    float e = warp_sum(epart[a]);
    if (lane == 0 && a < na) Ei[a0 + a] = e + ns.b1[0];
  }
  for (int n0 = 0; n0 < sp.Ndes; n0 += 64) {
    const int nu0 = n0 + lane, nu1 = nu0 + 32;
    const bool ok0 = nu0 < sp.Ndes, ok1 = nu1 < sp.Ndes;
    const float *w0p = ns.W0 + (ok0 ? nu0 : 0), *w1p = ns.W0 + (ok1 ? nu1 : 0);
    float acc0[GNEP_TILE], acc1[GNEP_TILE];
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) { acc0[a] = 0.f; acc1[a] = 0.f; }
    for (int mu = 0; mu < sp.Nn; ++mu) fma16x2(acc0, acc1, w0p[mu * sp.ldW], w1p[mu * sp.ldW], Cm + mu * GNEP_TILE);
    if (ok0) {
      const float s = ns.qs[nu0];
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a) {
        float v = s * acc0[a];
        if (a < na) Ep[(size_t)(a0 + a) * sp.Ndes + nu0] = v;
        if (nu0 < sp.NR) EpR[nu0 * GNEP_TILE + a] = v;
      }
    }
    if (ok1) {
      const float s = ns.qs[nu1];
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a) {
        float v = s * acc1[a];
        if (a < na) Ep[(size_t)(a0 + a) * sp.Ndes + nu1] = v;
        if (nu1 < sp.NR) EpR[nu1 * GNEP_TILE + a] = v;
      }
    }
  }
  __syncwarp();
  const int TK = sp.T * sp.KRp;
  for (int o = lane; o < TK; o += 32) {
    int J = o / sp.KRp, k = o - J * sp.KRp;
    float acc[GNEP_TILE], dummy[GNEP_TILE];
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) { acc[a] = 0.f; dummy[a] = 0.f; }
    for (int n = 0; n < sp.NR; ++n) fma16x2(acc, dummy, cRs[(J * sp.NR + n) * sp.KRp + k], 0.f, EpR + n * GNEP_TILE);
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a)
      if (a < na) etil[(size_t)(a0 + a) * TK + o] = acc[a];
  }
}

// ------------------------------------------------------------------------------------------------
// a6: network backward with the mixed second derivatives (paper Eq.D1.6-D1.17, C3.8):
//   p = W0 (s o D);  dL/dw1 += e x + d1 p;  A = w1 (e d1 + d2 p) -> dL/db0;  dL/db1 += e
//   h = s o W0^T (w1 d2 p) = E'' D;   gbar = e E' + h
// A and Bc = w1 d1 are written per atom for the W0 contraction (k_gemm_w0).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(GNEP_WARPS * 32)
k_net_bwd(DevSpec sp, SpeciesMap sm, const float *__restrict__ theta, const float *__restrict__ qscale,
          const int *__restrict__ struct_s, const float *__restrict__ e_s, const float *__restrict__ scales,
          const float *__restrict__ x, const float *__restrict__ Ep, const float *__restrict__ D,
          float *__restrict__ Acoef, float *__restrict__ Bcoef, float *__restrict__ gbar,
          float *__restrict__ partialB) {
  extern __shared__ __align__(16) float smem[];
  const int t = species_of_block(sm.cta_base, sp.T, blockIdx.x);
  NetSmem ns;
  float *nxt = stage_net(sp, smem, theta, qscale, t, ns);
  const int nb = 2 * sp.Nn + 1;
  float *redB = nxt;                                      // [GNEP_WARPS][nb]
  const int nred = (GNEP_WARPS * nb + 3) & ~3;
  const int per_warp = (sp.Ndes + sp.Nn + 1) * GNEP_TILE;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float *sD = nxt + nred + warp * per_warp;               // [Ndes][16]
  float *Hc = sD + sp.Ndes * GNEP_TILE;                   // [Nn][16]
  float *se = Hc + sp.Nn * GNEP_TILE;                     // [16] per-atom energy seed
  float *myB = redB + warp * nb;
  __syncthreads();
  int a0, na;
  net_tile(sm, t, a0, na);
  if (na <= 0) {
    for (int i = lane; i < nb; i += 32) myB[i] = 0.f;
  } else {
    if (lane < GNEP_TILE) se[lane] = lane < na ? scales[0] * e_s[struct_s[a0 + lane]] : 0.f;
    stage_rows_t(sD, D, ns.qs, a0, na, sp.Ndes, lane);
    __syncwarp();
    float e[GNEP_TILE], esum = 0.f;
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) { e[a] = se[a]; esum += e[a]; }
    for (int m0 = 0; m0 < sp.Nn; m0 += 64) {
      const int mu0 = m0 + lane, mu1 = mu0 + 32;
      const bool ok0 = mu0 < sp.Nn, ok1 = mu1 < sp.Nn;
      const float *w0p = ns.W0 + (ok0 ? mu0 : 0) * sp.ldW, *w1p = ns.W0 + (ok1 ? mu1 : 0) * sp.ldW;
      float p0[GNEP_TILE], p1[GNEP_TILE];
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a) { p0[a] = 0.f; p1[a] = 0.f; }
      for (int nu = 0; nu < sp.Ndes; ++nu) fma16x2(p0, p1, w0p[nu], w1p[nu], sD + nu * GNEP_TILE);
#pragma unroll
      for (int h2 = 0; h2 < 2; ++h2) {
        const int mu = h2 ? mu1 : mu0;
        if (h2 ? ok1 : ok0) {
          const float w1 = ns.w1[mu];
          float gw1 = 0.f, gb0 = 0.f;
#pragma unroll
          for (int a = 0; a < GNEP_TILE; ++a) {
            const float pv = h2 ? p1[a] : p0[a];
            float xv = a < na ? x[(size_t)(a0 + a) * sp.Nn + mu] : 0.f;
            float d1 = 1.f - xv * xv, d2 = -2.f * xv * d1;
            gw1 += e[a] * xv + d1 * pv;
            float A = w1 * (e[a] * d1 + d2 * pv);
            gb0 += A;
            if (a < na) {
              Acoef[(size_t)(a0 + a) * sp.Nn + mu] = A;
              Bcoef[(size_t)(a0 + a) * sp.Nn + mu] = w1 * d1;
            }
            Hc[mu * GNEP_TILE + a] = w1 * d2 * pv;
          }
          myB[mu] = gb0;
          myB[sp.Nn + mu] = gw1;
        }
      }
    }
    if (lane == 0) myB[2 * sp.Nn] = esum;
    __syncwarp();
    for (int n0 = 0; n0 < sp.Ndes; n0 += 64) {
      const int nu0 = n0 + lane, nu1 = nu0 + 32;
      const bool ok0 = nu0 < sp.Ndes, ok1 = nu1 < sp.Ndes;
      const float *w0p = ns.W0 + (ok0 ? nu0 : 0), *w1p = ns.W0 + (ok1 ? nu1 : 0);
      float h0[GNEP_TILE], h1[GNEP_TILE];
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a) { h0[a] = 0.f; h1[a] = 0.f; }
      for (int mu = 0; mu < sp.Nn; ++mu) fma16x2(h0, h1, w0p[mu * sp.ldW], w1p[mu * sp.ldW], Hc + mu * GNEP_TILE);
#pragma unroll
      for (int h2 = 0; h2 < 2; ++h2) {
        const int nu = h2 ? nu1 : nu0;
        if (h2 ? ok1 : ok0) {
          const float s = ns.qs[nu];
#pragma unroll
          for (int a = 0; a < GNEP_TILE; ++a)
            if (a < na) {
              size_t o = (size_t)(a0 + a) * sp.Ndes + nu;
              gbar[o] = e[a] * Ep[o] + s * (h2 ? h1[a] : h0[a]);
            }
        }
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < nb; i += blockDim.x) {
    float s = 0.f;
#pragma unroll
    for (int w = 0; w < GNEP_WARPS; ++w) s += redB[w * nb + i];
    partialB[(size_t)blockIdx.x * nb + i] = s;
  }
}

// ------------------------------------------------------------------------------------------------
// a6: dL/dW0[mu][nu] = sum_atoms A_mu G_nu + Bc_mu (s_nu D_nu)   (D1.9 + D1.14), one partial per K-chunk.
// Thread tile 4 mu x 8 nu (32 accumulators): per atom 6 LDS.128 for 64 FMA.  blockDim = ceil(Nn/4)*ceil(Ndes/8)
// threads rounded up to a warp (<= 384).  Shared rows are padded to multiples of 4 / 8 floats.
// ------------------------------------------------------------------------------------------------
#define GW_SUB 32
__host__ __device__ inline int gw_ldm(const DevSpec &sp) { return (sp.Nn + 3) & ~3; }
__host__ __device__ inline int gw_ldn(const DevSpec &sp) { return (sp.Ndes + 7) & ~7; }
__global__ void __launch_bounds__(384)
k_gemm_w0(DevSpec sp, SpeciesMap sm, const float *__restrict__ qscale, const float *__restrict__ q,
          const float *__restrict__ D, const float *__restrict__ Acoef, const float *__restrict__ Bcoef,
          float *__restrict__ partialW) {
  extern __shared__ __align__(16) float smem[];
  const int ldm = gw_ldm(sp), ldn = gw_ldn(sp);
  float *As = smem, *Bs = As + GW_SUB * ldm, *Gs = Bs + GW_SUB * ldm, *Ds = Gs + GW_SUB * ldn;
  const int t = species_of_block(sm.chunk_base, sp.T, blockIdx.x);
  const int c0 = sm.start[t] + (blockIdx.x - sm.chunk_base[t]) * sm.chunk_atoms[t];
  const int c1 = min(c0 + sm.chunk_atoms[t], sm.start[t + 1]);
  const int ngn = ldn >> 3, ngm = ldm >> 2;
  const int ng = threadIdx.x % ngn, mg = threadIdx.x / ngn;
  const bool act = mg < ngm;
  float acc[4][8];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;
  for (int s0 = c0; s0 < c1; s0 += GW_SUB) {
    const int ns_ = min(GW_SUB, c1 - s0);
    for (int x = threadIdx.x; x < GW_SUB * ldm; x += blockDim.x) {
      int at = x / ldm, mu = x - at * ldm;
      bool ok = at < ns_ && mu < sp.Nn;
      As[x] = ok ? Acoef[(size_t)(s0 + at) * sp.Nn + mu] : 0.f;
      Bs[x] = ok ? Bcoef[(size_t)(s0 + at) * sp.Nn + mu] : 0.f;
    }
    for (int x = threadIdx.x; x < GW_SUB * ldn; x += blockDim.x) {
      int at = x / ldn, nu = x - at * ldn;
      bool ok = at < ns_ && nu < sp.Ndes;
      float s = ok ? qscale[nu] : 0.f;
      Gs[x] = ok ? s * q[(size_t)(s0 + at) * sp.Ndes + nu] : 0.f;
      Ds[x] = ok ? s * D[(size_t)(s0 + at) * sp.Ndes + nu] : 0.f;
    }
    __syncthreads();
    if (act) {
      for (int at = 0; at < ns_; ++at) {
        const float4 a4 = *(const float4 *)(As + at * ldm + 4 * mg), b4 = *(const float4 *)(Bs + at * ldm + 4 * mg);
        const float4 g0 = *(const float4 *)(Gs + at * ldn + 8 * ng), g1 = *(const float4 *)(Gs + at * ldn + 8 * ng + 4);
        const float4 d0 = *(const float4 *)(Ds + at * ldn + 8 * ng), d1 = *(const float4 *)(Ds + at * ldn + 8 * ng + 4);
        const float av[4] = {a4.x, a4.y, a4.z, a4.w}, bv[4] = {b4.x, b4.y, b4.z, b4.w};
        const float gv[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
        const float dv[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 8; ++j) acc[i][j] += av[i] * gv[j] + bv[i] * dv[j];
      }
    }
    __syncthreads();
  }
  if (act) {
    float *out = partialW + (size_t)blockIdx.x * sp.Nn * sp.Ndes;
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        int mu = 4 * mg + i, nu = 8 * ng + j;
        if (mu < sp.Nn && nu < sp.Ndes) out[mu * sp.Ndes + nu] = acc[i][j];
      }
  }
}

// ------------------------------------------------------------------------------------------------
// a7 (radial): dL/dcR[I][J][n][k] = sum_{atoms of species I} gbar_n M1[J][k] + E'_n M2[J][k]
// (C1.3/C3.5 + C1.4-C1.5/C3.9 in moment-factored form: a rank-2 update per atom).  One partial per chunk,
// layout [n][J][k(KRp)].
// ------------------------------------------------------------------------------------------------
#define CR_SUB 64
__global__ void __launch_bounds__(256)
k_cgrad_radial(DevSpec sp, SpeciesMap sm, const float *__restrict__ gbar, const float *__restrict__ Ep,
               const float *__restrict__ M1, const float *__restrict__ M2, float *__restrict__ partialC) {
  extern __shared__ __align__(16) float smem[];
  const int TK = sp.T * sp.KRp;
  float *gb = smem, *ep = gb + CR_SUB * sp.NR, *m1 = ep + CR_SUB * sp.NR, *m2 = m1 + CR_SUB * TK;
  const int t = species_of_block(sm.chunk_base, sp.T, blockIdx.x);
  const int c0 = sm.start[t] + (blockIdx.x - sm.chunk_base[t]) * sm.chunk_atoms[t];
  const int c1 = min(c0 + sm.chunk_atoms[t], sm.start[t + 1]);
  const int O = sp.NR * TK;
  float acc[4] = {0.f, 0.f, 0.f, 0.f};
  for (int s0 = c0; s0 < c1; s0 += CR_SUB) {
    const int ns_ = min(CR_SUB, c1 - s0);
    for (int x = threadIdx.x; x < ns_ * sp.NR; x += 256) {
      int at = x / sp.NR, n = x - at * sp.NR;
      gb[x] = gbar[(size_t)(s0 + at) * sp.Ndes + n];
      ep[x] = Ep[(size_t)(s0 + at) * sp.Ndes + n];
    }
    for (int x = threadIdx.x; x < ns_ * TK; x += 256) {
      m1[x] = M1[(size_t)s0 * TK + x];
      m2[x] = M2[(size_t)s0 * TK + x];
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      int o = threadIdx.x + 256 * r;
      if (o < O) {
        int n = o / TK, jk = o - n * TK;
        float s = 0.f;
        for (int at = 0; at < ns_; ++at) s += gb[at * sp.NR + n] * m1[at * TK + jk] + ep[at * sp.NR + n] * m2[at * TK + jk];
        acc[r] += s;
      }
    }
    __syncthreads();
  }
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    int o = threadIdx.x + 256 * r;
    if (o < O) partialC[(size_t)blockIdx.x * O + o] = acc[r];
  }
}
