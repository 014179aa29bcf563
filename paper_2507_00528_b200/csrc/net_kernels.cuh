// net_kernels.cuh -- the "K = atoms" contraction of the radial coefficient gradient (row a7-radial of DESIGN.md).
// The network itself (rows a2, a6) lives in net_tc_kernels.cuh (tensor cores).
#pragma once
#include "common.cuh"
#include "net_tc_kernels.cuh"

// ------------------------------------------------------------------------------------------------
// a7 (radial): dL/dcR[I][J][n][k] = sum_{atoms of species I} gbar_n M1[J][k] + E'_n M2[J][k]
// (C1.3/C3.5 + C1.4-C1.5/C3.9 in moment-factored form: a rank-2 update per atom).  One partial per chunk,
// layout [n][J][k(KRp)].
// ------------------------------------------------------------------------------------------------
#define CR_SUB 64
__global__ void __launch_bounds__(256)
k_cgrad_radial(DevSpec sp, SpeciesMap sm, const float *__restrict__ gbar, const float *__restrict__ Ep,
               const float *__restrict__ M1, const float *__restrict__ M2, float *__restrict__ partialC) {
  extern __shared__ __align__(128) float smem[];
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
