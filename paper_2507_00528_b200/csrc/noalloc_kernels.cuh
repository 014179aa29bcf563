// noalloc_kernels.cuh -- kernel of gnep_loss_terms_noalloc (include/gnep.h): the loss terms of Eq.9-12 from
// caller-held predictions and references, a variant of k_struct_reduce (reduce_kernels.cuh) whose per-structure partial
// sums live in a fixed scratch array of the library instead of a per-batch allocation.
// One CTA per structure: fp64 sums of |F_i - Fref_i|^2 over the structure's atoms, the energy and virial residuals per
// atom (R18); the CTA that finishes last (ticket counter in the scratch) adds the per-structure parts in structure
// order -- fixed order, bit-reproducible -- and writes {L (without the L2 term), t_e, t_f, t_v}.
// Unit per-structure weights (Eq.10-12 as printed); a NULL reference drops its term (R39).
#pragma once
#include "../../include/gnep.h"
#include "common.cuh"
#include "reduce_kernels.cuh"

#define NOALLOC_MAX_STRUCTS GNEP_NOALLOC_MAX_STRUCTS               // structures per call (include/gnep.h: 8192)
#define NOALLOC_SCRATCH_DOUBLES (3 * NOALLOC_MAX_STRUCTS + 32)     // parts[S][3] + one 256-byte slot for the ticket

struct NoAllocLoss {
  int S;
  int loss_mode;
  double lam_e, lam_f, lam_v;
};

__global__ void __launch_bounds__(128)
k_loss_terms_noalloc(NoAllocLoss lc, const int *__restrict__ aoff /*[S+1]*/, const float *__restrict__ E /*[S]*/,
                     const float *__restrict__ F /*[N][3]*/, const float *__restrict__ W /*[S][6]*/,
                     const double *__restrict__ Eref, const double *__restrict__ Fref, const double *__restrict__ Wref,
                     double *scratch /*[NOALLOC_SCRATCH_DOUBLES]*/, float *__restrict__ terms /*[4]*/) {
  __shared__ double sh[4 * 4];
  __shared__ int last;
  double *parts = scratch;
  unsigned *ticket = (unsigned *)(scratch + 3 * NOALLOC_MAX_STRUCTS);
  const int s = blockIdx.x;
  const int b = aoff[s], e = aoff[s + 1];
  double v[1] = {0.0};
  if (Fref)
    for (int x = 3 * b + threadIdx.x; x < 3 * e; x += blockDim.x) {
      const double d = (double)F[x] - Fref[x];
      v[0] += d * d;
    }
  block_reduce_d<1>(v, sh);
  if (threadIdx.x == 0) {
    const double ns = (double)(e - b);
    double pe = 0.0, pv = 0.0;
    if (e > b) {
      if (Eref) { const double dE = ((double)E[s] - Eref[s]) / ns; pe = dE * dE; }
      if (Wref)
        for (int c = 0; c < 6; ++c) { const double dW = ((double)W[s * 6 + c] - Wref[s * 6 + c]) / ns; pv += dW * dW; }
    }
    parts[s * 3 + 0] = pe; parts[s * 3 + 1] = v[0]; parts[s * 3 + 2] = pv;
    __threadfence();                                               // parts visible before the ticket is taken
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double t[3] = {0.0, 0.0, 0.0};
  for (int i = threadIdx.x; i < lc.S; i += blockDim.x) { t[0] += __ldcg(parts + i * 3); t[1] += __ldcg(parts + i * 3 + 1); t[2] += __ldcg(parts + i * 3 + 2); }
  block_reduce_d<3>(t, sh);
  if (threadIdx.x == 0) {
    const double N = (double)aoff[lc.S];
    const double te = lc.S > 0 ? t[0] / lc.S : 0.0, tf = N > 0 ? t[1] / (3.0 * N) : 0.0, tv = lc.S > 0 ? t[2] / (6.0 * lc.S) : 0.0;
    const double L = lc.loss_mode == 0 ? lc.lam_e * te + lc.lam_f * tf + lc.lam_v * tv
                                       : lc.lam_e * sqrt(te) + lc.lam_f * sqrt(tf) + lc.lam_v * sqrt(tv);
    terms[0] = (float)L; terms[1] = (float)te; terms[2] = (float)tf; terms[3] = (float)tv;
    *ticket = 0u;                                                  // at rest the ticket is zero (the entry point also clears it)
  }
}
