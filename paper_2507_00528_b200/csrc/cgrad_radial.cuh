// cgrad_radial.cuh -- the radial expansion-coefficient gradient (row a7 of DESIGN.md) as a K = atoms contraction.
// The network itself (rows a2, a6) lives in net_tc_kernels.cuh (tensor cores).
#pragma once
#include "common.cuh"
#include "net_tc_kernels.cuh"

// ------------------------------------------------------------------------------------------------
// a7 (radial): dL/dcR[I][J][n][k] = sum_{atoms of species I} gbar_n M1[J][k] + E'_n M2[J][k]
// (C1.3/C3.5 + C1.4-C1.5/C3.9 in moment-factored form: a rank-2 update per atom).  One partial per chunk,
// layout [n][J][k(KRp)].
// A CTA stages CR_SUB atoms at a time (the NR radial columns of gbar and E', the moment rows) and contracts them with
// 4 n x 4 (J,k) register tiles: a "slice" of (NRp/4)(TKp/4) threads covers the whole output and takes every
// nslices-th atom of the stage (2 x 4 LDS.128 feed 32 FMA); the slices are summed through shared memory at the end.
// ------------------------------------------------------------------------------------------------
#define CR_SUB 128
#define CR_THREADS 256
__host__ __device__ inline int cr_nrp(const DevSpec &sp) { return (sp.NR + 3) & ~3; }
__host__ __device__ inline int cr_tkp(const DevSpec &sp) { return (sp.T * sp.KRp + 3) & ~3; }
__host__ __device__ inline size_t cgrad_radial_smem_bytes(const DevSpec &sp) {
  const size_t stage = (size_t)CR_SUB * 2 * (cr_nrp(sp) + cr_tkp(sp));
  const int per = (cr_nrp(sp) / 4) * (cr_tkp(sp) / 4);
  const size_t red = (size_t)(CR_THREADS / per) * cr_nrp(sp) * cr_tkp(sp);
  return sizeof(float) * (stage > red ? stage : red);
}
__global__ void __launch_bounds__(CR_THREADS)
k_cgrad_radial(DevSpec sp, SpeciesMap sm, const float *__restrict__ gbar, const float *__restrict__ Ep,
               const float *__restrict__ M1, const float *__restrict__ M2, float *__restrict__ partialC) {
  extern __shared__ __align__(128) float smem[];
  const int TK = sp.T * sp.KRp, NRp = cr_nrp(sp), TKp = cr_tkp(sp);
  float *gb = smem, *ep = gb + CR_SUB * NRp, *m1 = ep + CR_SUB * NRp, *m2 = m1 + CR_SUB * TKp;
  const int t = species_of_block(sm.chunk_base, sp.T, blockIdx.x);
  const int c0 = sm.start[t] + (blockIdx.x - sm.chunk_base[t]) * sm.chunk_atoms[t];
  const int c1 = min(c0 + sm.chunk_atoms[t], sm.start[t + 1]);
  const int nq = NRp >> 2, jq = TKp >> 2, per = nq * jq, nslices = CR_THREADS / per;
  const int slice = threadIdx.x / per, w = threadIdx.x - slice * per;
  const int n0 = 4 * (w / jq), j0 = 4 * (w - (w / jq) * jq);
  const bool on = slice < nslices;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  const int atA0 = threadIdx.x / NRp, nA0 = threadIdx.x - atA0 * NRp, datA = CR_THREADS / NRp, dnA = CR_THREADS - datA * NRp;
  const int atM0 = threadIdx.x / TKp, jkM0 = threadIdx.x - atM0 * TKp, datM = CR_THREADS / TKp, djkM = CR_THREADS - datM * TKp;
  for (int s0 = c0; s0 < c1; s0 += CR_SUB) {
    const int ns_ = min(CR_SUB, c1 - s0);
    {   // (at, n) and (at, jk) advance incrementally: no integer division per element (it cost as much as the FMAs)
      int at = atA0, n = nA0;
#pragma unroll 4
      for (int x = threadIdx.x; x < ns_ * NRp; x += CR_THREADS) {
        const bool ok = n < sp.NR;
        gb[x] = ok ? gbar[(size_t)(s0 + at) * sp.Ndes + n] : 0.f;
        ep[x] = ok ? Ep[(size_t)(s0 + at) * sp.Ndes + n] : 0.f;
        at += datA; n += dnA;
        if (n >= NRp) { n -= NRp; ++at; }
      }
      at = atM0; int jk = jkM0;
#pragma unroll 4
      for (int x = threadIdx.x; x < ns_ * TKp; x += CR_THREADS) {
        const bool ok = jk < TK;
        m1[x] = ok ? M1[(size_t)(s0 + at) * TK + jk] : 0.f;
        m2[x] = ok ? M2[(size_t)(s0 + at) * TK + jk] : 0.f;
        at += datM; jk += djkM;
        if (jk >= TKp) { jk -= TKp; ++at; }
      }
    }
    __syncthreads();
    if (on)
      for (int at = slice; at < ns_; at += nslices) {
        const float4 g4 = *(const float4 *)(gb + at * NRp + n0), e4 = *(const float4 *)(ep + at * NRp + n0);
        const float4 a4 = *(const float4 *)(m1 + at * TKp + j0), b4 = *(const float4 *)(m2 + at * TKp + j0);
        const float gv[4] = {g4.x, g4.y, g4.z, g4.w}, ev[4] = {e4.x, e4.y, e4.z, e4.w};
        const float av[4] = {a4.x, a4.y, a4.z, a4.w}, bv[4] = {b4.x, b4.y, b4.z, b4.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(gv[i], av[j], fmaf(ev[i], bv[j], acc[i][j]));
      }
    __syncthreads();
  }
  // slices -> one partial: red[slice][n][jk] over the staging buffers, summed in slice order
  float *red = smem;
  if (on)
#pragma unroll
    for (int i = 0; i < 4; ++i) *(float4 *)(red + ((size_t)slice * NRp + n0 + i) * TKp + j0) = make_float4(acc[i][0], acc[i][1], acc[i][2], acc[i][3]);
  __syncthreads();
  const int O = sp.NR * TK;
  for (int o = threadIdx.x; o < O; o += CR_THREADS) {
    const int n = o / TK, jk = o - n * TK;
    float s = 0.f;
    for (int sl = 0; sl < nslices; ++sl) s += red[((size_t)sl * NRp + n) * TKp + jk];
    partialC[(size_t)blockIdx.x * O + o] = s;
  }
}
