// net_small_kernels.cuh -- the per-atom tanh network (rows a2, a6) for SMALL batches, on plain FP32 FMAs.
//
// The tensor-core kernels of net_tc_kernels.cuh work on 128-atom tiles: a mini-batch of a few hundred atoms (the paper
// trains with batch size 1) gives them one or two tiles, and each launch then costs its fixed chain of TMEM
// allocation, weight staging and commit / wait round trips (13-15 us for a single tile, three launches per step).
// Here ONE WARP works on one atom (lane = neuron in the first contraction, lane = descriptor in the second), every
// species' network sits in shared memory (row stride odd: the column reads of the second contraction are
// conflict-free), and the backward kernel also forms the parameter-gradient partials, so a6 is one launch, not two.
// Same formulas as net_tc_kernels.cuh (Eq.D1.1, D1.5-D1.17, C3.8), plain fp32 dot products.
// Chosen by the host for small batches when the networks fit (gnep_api.cu); results agree with the tensor-core path to
// rounding and both are parity-tested against the oracle (tests/test_gpu_parity.py runs its core cases under both).
#pragma once
#include "common.cuh"
#include "net_tc_kernels.cuh"

#define NS_WARPS 4          // warps (= atoms in flight) per CTA
#define NS_ATOMS 4          // atoms per CTA (contiguous, one species): SpeciesMap.gw_atoms of a small batch

// W0 of one species (Nn x Ndes, row-major, contiguous at `net`) into shared memory with row stride ld; element
// x = mu * Ndes + nu is walked with incremental (mu, nu): no integer division in the loop, loads independent
__device__ __forceinline__ void ns_stage_w0(float *W0s, const float *__restrict__ net, int Nn, int Ndes, int ld) {
  const int nW = Nn * Ndes, step = NS_WARPS * 32;
  int mu = threadIdx.x / Ndes, nu = threadIdx.x - mu * Ndes;
  const int dmu = step / Ndes, dnu = step - dmu * Ndes;
#pragma unroll 4
  for (int x = threadIdx.x; x < nW; x += step) {
    W0s[mu * ld + nu] = net[x];
    mu += dmu; nu += dnu;
    if (nu >= Ndes) { nu -= Ndes; ++mu; }
  }
}
// sum_i w[i * ws] * v[i * vs], i < n, on four independent chains (the loads of a chain step do not wait for the FMAs)
__device__ __forceinline__ float ns_dot(const float *w, int ws, const float *v, int vs, int n) {
  float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
  int i = 0;
  for (; i + 3 < n; i += 4) {
    const float w0 = w[i * ws], w1 = w[(i + 1) * ws], w2 = w[(i + 2) * ws], w3 = w[(i + 3) * ws];
    const float v0 = v[i * vs], v1 = v[(i + 1) * vs], v2 = v[(i + 2) * vs], v3 = v[(i + 3) * vs];
    a0 = fmaf(w0, v0, a0); a1 = fmaf(w1, v1, a1); a2 = fmaf(w2, v2, a2); a3 = fmaf(w3, v3, a3);
  }
  for (; i < n; ++i) a0 = fmaf(w[i * ws], v[i * vs], a0);
  return (a0 + a1) + (a2 + a3);
}

// shared-memory floats of the forward kernel: cR[t] as [jk][16], the species' network, q_scale, per-warp rows
__host__ __device__ inline size_t net_small_fwd_floats(const DevSpec &sp) {
  return (size_t)sp.T * sp.KRp * 16 + (size_t)sp.Nn * sp.ldW + (size_t)(2 * sp.Nn + 1) + sp.Ndes +
         (size_t)NS_WARPS * (2 * sp.Ndes + sp.Nn);
}
// backward kernel: the species' network, w1, q_scale, per-warp rows sD, sG (Ndes each) and Hc, Av, Bv (Nn each), the W0
// gradient accumulator of the CTA and the cross-warp sums of the b0 / w1 / b1 partials
__host__ __device__ inline size_t net_small_bwd_floats(const DevSpec &sp) {
  return (size_t)sp.Nn * sp.ldW + (size_t)sp.Nn + sp.Ndes + (size_t)NS_WARPS * (2 * sp.Ndes + 3 * sp.Nn) +
         (size_t)sp.Nn * sp.Ndes + (size_t)NS_WARPS * (2 * sp.Nn + 1);
}

// ------------------------------------------------------------------------------------------------
// a2: x = tanh(W0 (s o q) + b0), E_i = w1.x + b1, E' = s o (C W0) with C = w1 (1 - x^2), etil = E'[0..NR) . cR
// A CTA owns a contiguous atom range of ONE species (SpeciesMap.gw_base / gw_atoms), its warps take one atom each.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NS_WARPS * 32)
k_net_small_fwd(DevSpec sp, SpeciesMap sm, const float *__restrict__ theta, const float *__restrict__ qscale,
                const float *__restrict__ q, float *__restrict__ xbuf, float *__restrict__ Ei, float *__restrict__ Ep,
                float *__restrict__ etil) {
  extern __shared__ __align__(128) float smem[];
  const int ld = sp.ldW, TK = sp.T * sp.KRp, nW = sp.Nn * sp.Ndes;
  float *cRs = smem;                                   // [jk = J*KRp + k][16]: cR[t][J][n][k], zero padded
  float *W0s = cRs + (size_t)TK * 16;                  // [mu][ld]
  float *bw = W0s + (size_t)sp.Nn * ld;                // [b0 (Nn) | w1 (Nn) | b1]
  float *qss = bw + (2 * sp.Nn + 1);                   // [Ndes]
  float *rows = qss + sp.Ndes + (size_t)(threadIdx.x >> 5) * (2 * sp.Ndes + sp.Nn);
  float *sq = rows, *Es = sq + sp.Ndes, *Cs = Es + sp.Ndes;   // per warp: s o q, E', C
  const int t = species_of_block(sm.gw_base, sp.T, blockIdx.x);
  const float *net = theta + sp.offNet + (size_t)t * sp.netSize;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int c0 = sm.start[t] + (blockIdx.x - sm.gw_base[t]) * sm.gw_atoms[t];
  const int c1 = min(c0 + sm.gw_atoms[t], sm.start[t + 1]);
  // the first atom's row is requested before the staging loops (it does not depend on them)
  float qpre[4] = {0.f, 0.f, 0.f, 0.f};
  if (c0 + warp < c1)
#pragma unroll
    for (int i = 0; i < 4; ++i) if (lane + 32 * i < sp.Ndes) qpre[i] = q[(size_t)(c0 + warp) * sp.Ndes + lane + 32 * i];
  ns_stage_w0(W0s, net, sp.Nn, sp.Ndes, ld);
  for (int x = threadIdx.x; x < 2 * sp.Nn + 1; x += blockDim.x) bw[x] = net[nW + x];
  for (int x = threadIdx.x; x < sp.Ndes; x += blockDim.x) qss[x] = qscale[x];
  for (int x = threadIdx.x; x < TK * 16; x += blockDim.x) {
    const int n = x & 15, jk = x >> 4, J = jk / sp.KRp, k = jk - J * sp.KRp;
    cRs[x] = (n < sp.NR && k < sp.KR) ? theta[(((size_t)t * sp.T + J) * sp.NR + n) * sp.KR + k] : 0.f;
  }
  __syncthreads();
  for (int a = c0 + warp; a < c1; a += NS_WARPS) {
#pragma unroll
    for (int i = 0; i < 4; ++i) if (lane + 32 * i < sp.Ndes) sq[lane + 32 * i] = qpre[i] * qss[lane + 32 * i];
    if (a + NS_WARPS < c1)
#pragma unroll
      for (int i = 0; i < 4; ++i) if (lane + 32 * i < sp.Ndes) qpre[i] = q[(size_t)(a + NS_WARPS) * sp.Ndes + lane + 32 * i];
    __syncwarp();
    float eacc = 0.f;
    for (int mu = lane; mu < sp.Nn; mu += 32) {          // first contraction: lane = neuron (row of W0, odd stride)
      const float z = bw[mu] + ns_dot(W0s + (size_t)mu * ld, 1, sq, 1, sp.Ndes);
      const float xv = tanh_fast(z), w1 = bw[sp.Nn + mu];
      xbuf[xt_off(a, mu, sp.NnS)] = xv;
      eacc = fmaf(w1, xv, eacc);
      Cs[mu] = w1 * (1.f - xv * xv);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) eacc += __shfl_xor_sync(0xffffffffu, eacc, o);
    if (lane == 0) Ei[a] = eacc + bw[2 * sp.Nn];
    __syncwarp();
    for (int nu = lane; nu < sp.Ndes; nu += 32) {        // second contraction: lane = descriptor (column of W0)
      const float e = ns_dot(W0s + nu, ld, Cs, 1, sp.Nn) * qss[nu];
      Ep[(size_t)a * sp.Ndes + nu] = e;
      Es[nu] = e;
    }
    __syncwarp();
    for (int jk = lane; jk < TK; jk += 32)               // etil[J][k] = sum_n E'_n cR[t][J][n][k]  (input of the radial force pass)
      etil[(size_t)a * TK + jk] = ns_dot(cRs + (size_t)jk * 16, 1, Es, 1, sp.NR);
    __syncwarp();
  }
}

// ------------------------------------------------------------------------------------------------
// a6, one launch: p = W0 (s o D), Hc = w1 d2 p, h = s o (Hc W0), gbar = e E' + h  (d1 = 1 - x^2, d2 = -2 x d1, D1.6, C3.8)
// and the parameter-gradient partials of this CTA's atoms (D1.7-D1.17):
//   dL/dW0 = sum A (x) G + Bc (x) sD,  dL/db0 = sum A,  dL/dw1 = sum V,  dL/db1 = sum e,
//   G = s o q, sD = s o D, A = w1 (e d1 + d2 p), Bc = w1 d1, V = e x + d1 p, e = s_e e_struct.
// Same atom ranges as the forward kernel; after a round (one atom per warp) all threads add the round's rank-2 updates to
// the CTA's W0-gradient accumulator in shared memory (element y = tid + 128 i).  One partial row per CTA, summed in row
// order by k_grad_reduce.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NS_WARPS * 32)
k_net_small_bwd(DevSpec sp, SpeciesMap sm, const float *__restrict__ theta, const float *__restrict__ qscale,
                const float *__restrict__ q, const float *__restrict__ D, const float *__restrict__ xbuf,
                const float *__restrict__ Ep, const int *__restrict__ struct_s, const float *__restrict__ e_s,
                const float *__restrict__ scales, float *__restrict__ gbar, float *__restrict__ partialW,
                float *__restrict__ partialB) {
  extern __shared__ __align__(128) float smem[];
  const int ld = sp.ldW, nW = sp.Nn * sp.Ndes, nrow = 2 * sp.Ndes + 3 * sp.Nn;
  float *W0s = smem;                                   // [mu][ld] of this CTA's species
  float *w1s = W0s + (size_t)sp.Nn * ld;               // [Nn]
  float *qss = w1s + sp.Nn;                            // [Ndes]
  float *rows0 = qss + sp.Ndes;                        // per warp: sD | sG | Hc | Av | Bv
  float *accW = rows0 + (size_t)NS_WARPS * nrow;       // [Nn * Ndes]
  float *red = accW + nW;                              // [warp][b0 (Nn) | w1 (Nn) | b1]
  const int t = species_of_block(sm.gw_base, sp.T, blockIdx.x);
  const float *net = theta + sp.offNet + (size_t)t * sp.netSize;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int c0 = sm.start[t] + (blockIdx.x - sm.gw_base[t]) * sm.gw_atoms[t];
  const int c1 = min(c0 + sm.gw_atoms[t], sm.start[t + 1]);
  ns_stage_w0(W0s, net, sp.Nn, sp.Ndes, ld);
  for (int x = threadIdx.x; x < sp.Nn; x += blockDim.x) w1s[x] = net[nW + sp.Nn + x];
  for (int x = threadIdx.x; x < sp.Ndes; x += blockDim.x) qss[x] = qscale[x];
  for (int x = threadIdx.x; x < nW; x += blockDim.x) accW[x] = 0.f;
  __syncthreads();
  float *sD = rows0 + (size_t)warp * nrow, *sG = sD + sp.Ndes, *Hc = sG + sp.Ndes, *Av = Hc + sp.Nn, *Bv = Av + sp.Nn;
  const float se = scales[0];
  float accA[4] = {0.f, 0.f, 0.f, 0.f}, accV[4] = {0.f, 0.f, 0.f, 0.f}, acce = 0.f;   // neurons lane, lane + 32, ... (Nn <= 128)
  const int step = NS_WARPS * 32;
  const int mu_first = threadIdx.x / sp.Ndes, nu_first = threadIdx.x - mu_first * sp.Ndes;
  const int dmu = step / sp.Ndes, dnu = step - dmu * sp.Ndes;
  for (int r0 = c0; r0 < c1; r0 += NS_WARPS) {
    const int a = r0 + warp;
    if (a < c1) {
      const float e = se * e_s[struct_s[a]];
      acce += e;                                       // (every lane holds it; lane 0's copy is used)
      float xv[4], epv[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {                    // requested before the contractions that need them
        xv[i] = lane + 32 * i < sp.Nn ? xbuf[xt_off(a, lane + 32 * i, sp.NnS)] : 0.f;
        epv[i] = lane + 32 * i < sp.Ndes ? Ep[(size_t)a * sp.Ndes + lane + 32 * i] : 0.f;
      }
      for (int nu = lane; nu < sp.Ndes; nu += 32) {
        const float s = qss[nu];
        sD[nu] = D[(size_t)a * sp.Ndes + nu] * s;
        sG[nu] = q[(size_t)a * sp.Ndes + nu] * s;
      }
      __syncwarp();
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int mu = lane + 32 * i;
        if (mu < sp.Nn) {
          const float p = ns_dot(W0s + (size_t)mu * ld, 1, sD, 1, sp.Ndes), w1 = w1s[mu];
          const float d1 = 1.f - xv[i] * xv[i], d2 = -2.f * xv[i] * d1;
          const float A = w1 * (e * d1 + d2 * p);
          Hc[mu] = w1 * d2 * p; Av[mu] = A; Bv[mu] = w1 * d1;
          accA[i] += A;
          accV[i] += e * xv[i] + d1 * p;
        }
      }
      __syncwarp();
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int nu = lane + 32 * i;
        if (nu < sp.Ndes) gbar[(size_t)a * sp.Ndes + nu] = e * epv[i] + ns_dot(W0s + nu, ld, Hc, 1, sp.Nn) * qss[nu];
      }
    }
    __syncthreads();
    // the round's rank-2 updates to the elements this thread owns
    const int nw_on = min(NS_WARPS, c1 - r0);
    int mu = mu_first, nu = nu_first;
#pragma unroll 2
    for (int y = threadIdx.x; y < nW; y += step) {
      float s = accW[y];
#pragma unroll
      for (int w = 0; w < NS_WARPS; ++w) {
        if (w < nw_on) {
          const float *rw = rows0 + (size_t)w * nrow;   // sD | sG | Hc | Av | Bv of warp w's atom
          s = fmaf(rw[2 * sp.Ndes + sp.Nn + mu], rw[sp.Ndes + nu], fmaf(rw[2 * sp.Ndes + 2 * sp.Nn + mu], rw[nu], s));
        }
      }
      accW[y] = s;
      mu += dmu; nu += dnu;
      if (nu >= sp.Ndes) { nu -= sp.Ndes; ++mu; }
    }
    __syncthreads();
  }
  for (int y = threadIdx.x; y < nW; y += step) partialW[(size_t)blockIdx.x * nW + y] = accW[y];
  float *rd = red + (size_t)warp * (2 * sp.Nn + 1);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int mu = lane + 32 * i;
    if (mu < sp.Nn) { rd[mu] = accA[i]; rd[sp.Nn + mu] = accV[i]; }
  }
  if (lane == 0) rd[2 * sp.Nn] = acce;
  __syncthreads();
  for (int x = threadIdx.x; x < 2 * sp.Nn + 1; x += blockDim.x) {
    float s = 0.f;
    for (int w = 0; w < NS_WARPS; ++w) s += red[(size_t)w * (2 * sp.Nn + 1) + x];
    partialB[(size_t)blockIdx.x * (2 * sp.Nn + 1) + x] = s;
  }
}
