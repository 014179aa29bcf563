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
  float *G = nxt + ncr + (threadIdx.x >> 5) * per_warp;   // [Ndes][8]
  float *Cm = G + sp.Ndes * GNEP_TILE;                     // [Nn][8]
  float *EpR = Cm + sp.Nn * GNEP_TILE;                     // [NR][8]
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int a0 = sm.start[t] + ((blockIdx.x - sm.cta_base[t]) * GNEP_WARPS + (threadIdx.x >> 5)) * GNEP_TILE;
  const int na = min(GNEP_TILE, sm.start[t + 1] - a0);
  if (na <= 0) return;
  for (int a = 0; a < GNEP_TILE; ++a)
    for (int nu = lane; nu < sp.Ndes; nu += 32)
      G[nu * GNEP_TILE + a] = a < na ? ns.qs[nu] * q[(size_t)(a0 + a) * sp.Ndes + nu] : 0.f;
  __syncwarp();
  float epart[GNEP_TILE];
#pragma unroll
  for (int a = 0; a < GNEP_TILE; ++a) epart[a] = 0.f;
  for (int mu = lane; mu < sp.Nn; mu += 32) {
    float acc[GNEP_TILE];
    const float b = ns.b0[mu];
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) acc[a] = b;
    const float *w = ns.W0 + mu * sp.ldW;
    for (int nu = 0; nu < sp.Ndes; ++nu) {
      float wv = w[nu];
      float4 g0 = *(const float4 *)(G + nu * GNEP_TILE), g1 = *(const float4 *)(G + nu * GNEP_TILE + 4);
      acc[0] += wv * g0.x; acc[1] += wv * g0.y; acc[2] += wv * g0.z; acc[3] += wv * g0.w;
      acc[4] += wv * g1.x; acc[5] += wv * g1.y; acc[6] += wv * g1.z; acc[7] += wv * g1.w;
    }
    const float w1 = ns.w1[mu];
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) {
      float xv = tanhf(acc[a]);
      if (a < na) xout[(size_t)(a0 + a) * sp.Nn + mu] = xv;
      Cm[mu * GNEP_TILE + a] = w1 * (1.f - xv * xv);
      epart[a] += w1 * xv;
    }
  }
  __syncwarp();
#pragma unroll
  for (int a = 0; a < GNEP_TILE; ++a) {
    float e = warp_sum(epart[a]);
    if (lane == 0 && a < na) Ei[a0 + a] = e + ns.b1[0];
  }
  for (int nu = lane; nu < sp.Ndes; nu += 32) {
    float acc[GNEP_TILE];
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) acc[a] = 0.f;
    for (int mu = 0; mu < sp.Nn; ++mu) {
      float wv = ns.W0[mu * sp.ldW + nu];
      float4 c0 = *(const float4 *)(Cm + mu * GNEP_TILE), c1 = *(const float4 *)(Cm + mu * GNEP_TILE + 4);
      acc[0] += wv * c0.x; acc[1] += wv * c0.y; acc[2] += wv * c0.z; acc[3] += wv * c0.w;
      acc[4] += wv * c1.x; acc[5] += wv * c1.y; acc[6] += wv * c1.z; acc[7] += wv * c1.w;
    }
    const float s = ns.qs[nu];
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) {
      float v = s * acc[a];
      if (a < na) Ep[(size_t)(a0 + a) * sp.Ndes + nu] = v;
      if (nu < sp.NR) EpR[nu * GNEP_TILE + a] = v;
    }
  }
  __syncwarp();
  const int TK = sp.T * sp.KRp;
  for (int o = lane; o < TK; o += 32) {
    int J = o / sp.KRp, k = o - J * sp.KRp;
    float acc[GNEP_TILE];
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) acc[a] = 0.f;
    for (int n = 0; n < sp.NR; ++n) {
      float cv = cRs[(J * sp.NR + n) * sp.KRp + k];
      float4 e0 = *(const float4 *)(EpR + n * GNEP_TILE), e1 = *(const float4 *)(EpR + n * GNEP_TILE + 4);
      acc[0] += cv * e0.x; acc[1] += cv * e0.y; acc[2] += cv * e0.z; acc[3] += cv * e0.w;
      acc[4] += cv * e1.x; acc[5] += cv * e1.y; acc[6] += cv * e1.z; acc[7] += cv * e1.w;
    }
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
  const int per_warp = (sp.Ndes + sp.Nn) * GNEP_TILE;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float *sD = nxt + nred + warp * per_warp;               // [Ndes][8]
  float *Hc = sD + sp.Ndes * GNEP_TILE;                   // [Nn][8]
  float *myB = redB + warp * nb;
  __syncthreads();
  const int a0 = sm.start[t] + ((blockIdx.x - sm.cta_base[t]) * GNEP_WARPS + warp) * GNEP_TILE;
  const int na = min(GNEP_TILE, sm.start[t + 1] - a0);
  if (na <= 0) {
    for (int i = lane; i < nb; i += 32) myB[i] = 0.f;
  } else {
    float e[GNEP_TILE];
    const float se = scales[0];
    float esum = 0.f;
#pragma unroll
    for (int a = 0; a < GNEP_TILE; ++a) { e[a] = a < na ? se * e_s[struct_s[a0 + a]] : 0.f; esum += e[a]; }
    for (int a = 0; a < GNEP_TILE; ++a)
      for (int nu = lane; nu < sp.Ndes; nu += 32)
        sD[nu * GNEP_TILE + a] = a < na ? ns.qs[nu] * D[(size_t)(a0 + a) * sp.Ndes + nu] : 0.f;
    __syncwarp();
    for (int mu = lane; mu < sp.Nn; mu += 32) {
      float p[GNEP_TILE];
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a) p[a] = 0.f;
      const float *w = ns.W0 + mu * sp.ldW;
      for (int nu = 0; nu < sp.Ndes; ++nu) {
        float wv = w[nu];
        float4 g0 = *(const float4 *)(sD + nu * GNEP_TILE), g1 = *(const float4 *)(sD + nu * GNEP_TILE + 4);
        p[0] += wv * g0.x; p[1] += wv * g0.y; p[2] += wv * g0.z; p[3] += wv * g0.w;
        p[4] += wv * g1.x; p[5] += wv * g1.y; p[6] += wv * g1.z; p[7] += wv * g1.w;
      }
      const float w1 = ns.w1[mu];
      float gw1 = 0.f, gb0 = 0.f;
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a) {
        float xv = a < na ? x[(size_t)(a0 + a) * sp.Nn + mu] : 0.f;
        float d1 = 1.f - xv * xv, d2 = -2.f * xv * d1;
        gw1 += e[a] * xv + d1 * p[a];
        float A = w1 * (e[a] * d1 + d2 * p[a]);
        gb0 += A;
        if (a < na) {
          Acoef[(size_t)(a0 + a) * sp.Nn + mu] = A;
          Bcoef[(size_t)(a0 + a) * sp.Nn + mu] = w1 * d1;
        }
        Hc[mu * GNEP_TILE + a] = w1 * d2 * p[a];
      }
      myB[mu] = gb0;
      myB[sp.Nn + mu] = gw1;
    }
    if (lane == 0) myB[2 * sp.Nn] = esum;
    __syncwarp();
    for (int nu = lane; nu < sp.Ndes; nu += 32) {
      float h[GNEP_TILE];
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a) h[a] = 0.f;
      for (int mu = 0; mu < sp.Nn; ++mu) {
        float wv = ns.W0[mu * sp.ldW + nu];
        float4 c0 = *(const float4 *)(Hc + mu * GNEP_TILE), c1 = *(const float4 *)(Hc + mu * GNEP_TILE + 4);
        h[0] += wv * c0.x; h[1] += wv * c0.y; h[2] += wv * c0.z; h[3] += wv * c0.w;
        h[4] += wv * c1.x; h[5] += wv * c1.y; h[6] += wv * c1.z; h[7] += wv * c1.w;
      }
      const float s = ns.qs[nu];
#pragma unroll
      for (int a = 0; a < GNEP_TILE; ++a)
        if (a < na) {
          size_t o = (size_t)(a0 + a) * sp.Ndes + nu;
          gbar[o] = e[a] * Ep[o] + s * h[a];
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
// 256 threads = 16 (mu groups) x 16 (nu groups); thread tile mu = mg+16 i, nu = ng+16 j.
// ------------------------------------------------------------------------------------------------
#define GW_SUB 32
__global__ void __launch_bounds__(256)
k_gemm_w0(DevSpec sp, SpeciesMap sm, const float *__restrict__ qscale, const float *__restrict__ q,
          const float *__restrict__ D, const float *__restrict__ Acoef, const float *__restrict__ Bcoef,
          float *__restrict__ partialW) {
  extern __shared__ __align__(16) float smem[];
  float *As = smem, *Bs = As + GW_SUB * sp.Nn, *Gs = Bs + GW_SUB * sp.Nn, *Ds = Gs + GW_SUB * sp.Ndes;
  const int t = species_of_block(sm.chunk_base, sp.T, blockIdx.x);
  const int c0 = sm.start[t] + (blockIdx.x - sm.chunk_base[t]) * sm.chunk_atoms[t];
  const int c1 = min(c0 + sm.chunk_atoms[t], sm.start[t + 1]);
  const int mg = threadIdx.x & 15, ng = threadIdx.x >> 4;
  float acc[8][6];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 6; ++j) acc[i][j] = 0.f;
  for (int s0 = c0; s0 < c1; s0 += GW_SUB) {
    const int ns_ = min(GW_SUB, c1 - s0);
    for (int x = threadIdx.x; x < GW_SUB * sp.Nn; x += 256) {
      bool ok = x < ns_ * sp.Nn;
      As[x] = ok ? Acoef[(size_t)s0 * sp.Nn + x] : 0.f;
      Bs[x] = ok ? Bcoef[(size_t)s0 * sp.Nn + x] : 0.f;
    }
    for (int x = threadIdx.x; x < GW_SUB * sp.Ndes; x += 256) {
      bool ok = x < ns_ * sp.Ndes;
      float s = qscale[x % sp.Ndes];
      Gs[x] = ok ? s * q[(size_t)s0 * sp.Ndes + x] : 0.f;
      Ds[x] = ok ? s * D[(size_t)s0 * sp.Ndes + x] : 0.f;
    }
    __syncthreads();
    for (int at = 0; at < ns_; ++at) {
      float av[8], bv[8], gv[6], dv[6];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        int mu = mg + 16 * i;
        av[i] = mu < sp.Nn ? As[at * sp.Nn + mu] : 0.f;
        bv[i] = mu < sp.Nn ? Bs[at * sp.Nn + mu] : 0.f;
      }
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        int nu = ng + 16 * j;
        gv[j] = nu < sp.Ndes ? Gs[at * sp.Ndes + nu] : 0.f;
        dv[j] = nu < sp.Ndes ? Ds[at * sp.Ndes + nu] : 0.f;
      }
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 6; ++j) acc[i][j] += av[i] * gv[j] + bv[i] * dv[j];
    }
    __syncthreads();
  }
  float *out = partialW + (size_t)blockIdx.x * sp.Nn * sp.Ndes;
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      int mu = mg + 16 * i, nu = ng + 16 * j;
      if (mu < sp.Nn && nu < sp.Ndes) out[mu * sp.Ndes + nu] = acc[i][j];
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
