// net_small_kernels.cuh -- the per-atom tanh network (rows a2, a6) for SMALL batches, on plain FP32 FMAs.
//
// The tensor-core kernels of net_tc_kernels.cuh work on 128-atom tiles: a mini-batch of a few hundred atoms (the paper
// trains with batch size 1) gives them one or two tiles, and each launch then costs its fixed chain of TMEM
// allocation, weight staging and commit / wait round trips (13-15 us for a single tile, three launches per step).
// Here a group of 128 THREADS works on one atom (thread = neuron in the first contraction, thread = descriptor in the
// second: every dot product of the two contractions runs at once), a CTA holds four such groups and one species' network
// in shared memory (row stride odd: row and column reads are both conflict-free), and the backward kernel also forms the
// parameter-gradient partials, so a6 is one launch, not two.  With so few warps per SM these kernels are bound by the
// number of instructions a warp executes one after the other: the mapping keeps that number small.
// Same formulas as net_tc_kernels.cuh (Eq.D1.1, D1.5-D1.17, C3.8), plain fp32 dot products.
// Chosen by the host for small batches when the networks fit (gnep_api.cu); results agree with the tensor-core path to
// rounding and both are parity-tested against the oracle (tests/test_gpu_parity.py runs its core cases under both).
#pragma once
#include "common.cuh"
#include "net_tc_kernels.cuh"

#define NS_GROUP 128        // threads per atom
#define NS_ATOMS 4          // atoms per CTA and round (contiguous, one species): SpeciesMap.gw_atoms of a small batch
#define NS_THREADS (NS_GROUP * NS_ATOMS)

// species t and atom range [c0, c1) of CTA `bid` (SpeciesMap.gw_base / gw_atoms / start) with STATIC indices into the
// kernel-parameter struct: a dynamic index makes the compiler copy the struct to local memory (a fifth of the
// instructions of these short kernels)
__device__ __forceinline__ void ns_range(const SpeciesMap &sm, int T, int bid, int &t, int &c0, int &c1) {
  int base = sm.gw_base[0], start = sm.start[0], end = sm.start[1], ga = sm.gw_atoms[0];
  t = 0;
#pragma unroll
  for (int i = 1; i < GNEP_MAX_SPECIES_C; ++i)
    if (i < T && bid >= sm.gw_base[i]) { t = i; base = sm.gw_base[i]; start = sm.start[i]; end = sm.start[i + 1]; ga = sm.gw_atoms[i]; }
  c0 = start + (bid - base) * ga;
  c1 = min(c0 + ga, end);
}

// W0 of one species (Nn x Ndes, row-major, contiguous at `net`) into shared memory with row stride ld; element
// x = mu * Ndes + nu is walked with incremental (mu, nu): no integer division in the loop, loads independent
__device__ __forceinline__ void ns_stage_w0(float *W0s, const float *__restrict__ net, int Nn, int Ndes, int ld) {
  const int nW = Nn * Ndes;
  int mu = threadIdx.x / Ndes, nu = threadIdx.x - mu * Ndes;
  const int dmu = NS_THREADS / Ndes, dnu = NS_THREADS - dmu * Ndes;
#pragma unroll 4
  for (int x = threadIdx.x; x < nW; x += NS_THREADS) {
    W0s[mu * ld + nu] = net[x];
    mu += dmu; nu += dnu;
    if (nu >= Ndes) { nu -= Ndes; ++mu; }
  }
}
// sum_i w[i * ws] * v[i], i < n, on four independent chains (the loads of a chain step do not wait for the FMAs)
__device__ __forceinline__ float ns_dot(const float *w, int ws, const float *v, int n) {
  float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
  int i = 0;
  for (; i + 3 < n; i += 4, w += 4 * ws) {
    const float w0 = w[0], w1 = w[ws], w2 = w[2 * ws], w3 = w[3 * ws];
    const float4 v4 = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
    a0 = fmaf(w0, v4.x, a0); a1 = fmaf(w1, v4.y, a1); a2 = fmaf(w2, v4.z, a2); a3 = fmaf(w3, v4.w, a3);
  }
  for (; i < n; ++i, w += ws) a0 = fmaf(w[0], v[i], a0);
  return (a0 + a1) + (a2 + a3);
}

// shared-memory floats of the forward kernel: cR[t] as [jk][16], the species' network, q_scale, per-atom rows; with the
// descriptor contraction fused in (warp-tile angular path): cA[t], and per atom the A1 block, the M1 row, S and q
__host__ __device__ inline size_t net_small_fwd_floats(const DevSpec &sp) {
  return (size_t)sp.T * sp.KRp * 16 + (size_t)sp.Nn * sp.ldW + (size_t)(2 * sp.Nn + 1) + sp.Ndes +
         (size_t)NS_ATOMS * (2 * sp.Ndes + sp.Nn + 4) + (size_t)sp.T * sp.NA * sp.KAp +
         (size_t)NS_ATOMS * (sp.T * sp.KAp * 24 + sp.T * sp.KRp + sp.NA * 24 + sp.Ndes);
}
// backward kernel: the species' network, w1, q_scale, per-atom rows sD, sG (Ndes each) and Hc, Av, Bv (Nn each), the W0
// gradient accumulator of the CTA and the cross-group sums of the b0 / w1 / b1 partials
__host__ __device__ inline size_t net_small_bwd_floats(const DevSpec &sp) {
  return (size_t)sp.Nn * sp.ldW + (size_t)sp.Nn + sp.Ndes + (size_t)NS_ATOMS * (2 * sp.Ndes + 3 * sp.Nn) +
         (size_t)sp.Nn * sp.Ndes + (size_t)NS_ATOMS * (2 * sp.Nn + 1) +
         (size_t)NS_ATOMS * (2 * sp.NR + 2 * sp.T * sp.KRp) + (size_t)sp.NR * sp.T * sp.KRp;   // radial c-gradient rows and accumulator
}

// ------------------------------------------------------------------------------------------------
// a2: x = tanh(W0 (s o q) + b0), E_i = w1.x + b1, E' = s o (C W0) with C = w1 (1 - x^2), etil = E'[0..NR) . cR
// A CTA owns a contiguous atom range of ONE species (SpeciesMap.gw_base / gw_atoms), NS_ATOMS atoms per round.
// With A1 != nullptr (angular warp-tile path, l_max <= 4) the per-epoch descriptor contraction a1 is done here too, from
// the resident geometry moments (angular_warp_kernels.cuh, k_angw_S): q_n = cR.M1 (Eq.5-6), S_nlm = cA.A1 (Eq.8, thread
// = (n, lm)), q_nl = sum_m C_lm S^2 (Eq.7), the 4-body (R14) and 5-body (R41) terms; q and S are written for the later
// kernels and the network reads q from shared memory: one launch instead of two.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NS_THREADS)
k_net_small_fwd(DevSpec sp, SpeciesMap sm, const float *__restrict__ theta, const float *__restrict__ qscale,
                float *q, float *__restrict__ xbuf, float *__restrict__ Ei, float *__restrict__ Ep,
                float *__restrict__ etil, const float *__restrict__ A1, const float *__restrict__ M1, float *__restrict__ S) {
  extern __shared__ __align__(128) float smem[];
  const int ld = sp.ldW, TK = sp.T * sp.KRp, nW = sp.Nn * sp.Ndes, nrow = 2 * sp.Ndes + sp.Nn + 4;
  const int grp = threadIdx.x >> 7, tig = threadIdx.x & (NS_GROUP - 1);
  float *cRs = smem;                                   // [jk = J*KRp + k][16]: cR[t][J][n][k], zero padded
  float *W0s = cRs + (size_t)TK * 16;                  // [mu][ld]
  float *bw = W0s + (size_t)sp.Nn * ld;                // [b0 (Nn) | w1 (Nn) | b1]
  float *qss = bw + (2 * sp.Nn + 1);                   // [Ndes]
  float *sq = qss + sp.Ndes + (size_t)grp * nrow, *Es = sq + sp.Ndes, *Cs = Es + sp.Ndes, *ep4 = Cs + sp.Nn;   // per atom: s o q, E', C, E partials
  const bool fuse = A1 != nullptr;
  const int nA1 = sp.T * sp.KAp * 24, nS = sp.NA * 24, ndr = nA1 + TK + nS + sp.Ndes;
  float *cAs = qss + sp.Ndes + (size_t)NS_ATOMS * nrow;            // [J][n][k(KAp)] of this species, zero padded
  float *A1s = cAs + (size_t)sp.T * sp.NA * sp.KAp + (size_t)grp * ndr, *m1s = A1s + nA1, *Ss = m1s + TK, *qrow = Ss + nS;
  int t, c0, c1;
  ns_range(sm, sp.T, blockIdx.x, t, c0, c1);
  const float *net = theta + sp.offNet + (size_t)t * sp.netSize;
  // the first atom's row is requested before the staging loops (it does not depend on them)
  float qv = (!fuse && c0 + grp < c1 && tig < sp.Ndes) ? q[(size_t)(c0 + grp) * sp.Ndes + tig] : 0.f;
  if (fuse) {
    if (c0 + grp < c1) {                                 // the first atom's moments: requested before the staging loops too
      const int a = c0 + grp;
      for (int x = tig; x < nA1; x += NS_GROUP) A1s[x] = A1[(size_t)a * nA1 + x];
      for (int x = tig; x < TK; x += NS_GROUP) m1s[x] = M1[(size_t)a * TK + x];
    }
    for (int x = threadIdx.x; x < sp.T * sp.NA * sp.KAp; x += NS_THREADS) {
      const int k = x % sp.KAp, jn = x / sp.KAp;         // jn = J * NA + n
      cAs[x] = k < sp.KA ? theta[sp.offA + ((size_t)t * sp.T * sp.NA + jn) * sp.KA + k] : 0.f;
    }
  }
  ns_stage_w0(W0s, net, sp.Nn, sp.Ndes, ld);
  for (int x = threadIdx.x; x < 2 * sp.Nn + 1; x += NS_THREADS) bw[x] = net[nW + x];
  for (int x = threadIdx.x; x < sp.Ndes; x += NS_THREADS) qss[x] = qscale[x];
  for (int x = threadIdx.x; x < TK * 16; x += NS_THREADS) {
    const int n = x & 15, jk = x >> 4, J = jk / sp.KRp, k = jk - J * sp.KRp;
    cRs[x] = (n < sp.NR && k < sp.KR) ? theta[(((size_t)t * sp.T + J) * sp.NR + n) * sp.KR + k] : 0.f;
  }
  __syncthreads();
  for (int r0 = c0; r0 < c1; r0 += NS_ATOMS) {
    const int a = r0 + grp;
    const bool on = a < c1;
    if (fuse) {
      if (on && r0 > c0) {
        for (int x = tig; x < nA1; x += NS_GROUP) A1s[x] = A1[(size_t)a * nA1 + x];
        for (int x = tig; x < TK; x += NS_GROUP) m1s[x] = M1[(size_t)a * TK + x];
      }
      __syncthreads();
      if (on) {
        for (int y = tig; y < nS; y += NS_GROUP) {       // S[n][lm] = sum_{J,k} cA[t][J][n][k] A1[J][k][lm]
          const int n = y / 24, lm = y - n * 24;
          float s0 = 0.f, s1 = 0.f;
          for (int J = 0; J < sp.T; ++J) {
            const float *c = cAs + (size_t)(J * sp.NA + n) * sp.KAp, *m = A1s + (size_t)J * sp.KAp * 24 + lm;
            for (int k = 0; k < sp.KAp; k += 2) { s0 = fmaf(c[k], m[k * 24], s0); s1 = fmaf(c[k + 1], m[(k + 1) * 24], s1); }
          }
          Ss[y] = s0 + s1;
          S[(size_t)a * nS + y] = s0 + s1;
        }
        if (tig < sp.NR) {                               // q_n = sum_{J,k} cR[t][J][n][k] M1[J][k]
          float s0 = 0.f;
          for (int jk = 0; jk < TK; ++jk) s0 = fmaf(cRs[jk * 16 + tig], m1s[jk], s0);
          qrow[tig] = s0;
        }
      }
      __syncthreads();
      if (on) {
        const int nl = sp.NA * sp.L;
        if (tig < nl) {                                  // q_nl = sum_m C_lm S_nlm^2, descriptor index NR + (l-1) NA + n
          const int l = tig / sp.NA + 1, n = tig - (l - 1) * sp.NA;
          float v = 0.f;
          for (int lm = l * l - 1; lm < l * l + 2 * l; ++lm) { const float sv = Ss[n * 24 + lm]; v = fmaf(0.5f * c_C2[lm] * sv, sv, v); }
          qrow[sp.NR + tig] = v;
        } else if (sp.use4 && tig < nl + sp.NA) {
          qrow[sp.NR + tig] = GNEP_KAPPA4 * p4_value(Ss + (tig - nl) * 24 + 3);
        } else if (sp.use5 && tig < nl + (sp.use4 + 1) * sp.NA) {
          qrow[sp.NR + tig] = p5_value(Ss + (tig - nl - sp.use4 * sp.NA) * 24);
        }
      }
      __syncthreads();
      if (on && tig < sp.Ndes) { const float qx = qrow[tig]; q[(size_t)a * sp.Ndes + tig] = qx; sq[tig] = qx * qss[tig]; }
    } else {
      if (on && tig < sp.Ndes) sq[tig] = qv * qss[tig];
      if (a + NS_ATOMS < c1 && tig < sp.Ndes) qv = q[(size_t)(a + NS_ATOMS) * sp.Ndes + tig];
    }
    __syncthreads();
    float e = 0.f;
    if (on && tig < sp.Nn) {                             // first contraction: thread = neuron (row of W0, odd stride)
      const float z = bw[tig] + ns_dot(W0s + (size_t)tig * ld, 1, sq, sp.Ndes);
      const float xv = tanh_fast(z), w1 = bw[sp.Nn + tig];
      xbuf[xt_off(a, tig, sp.NnS)] = xv;
      e = w1 * xv;
      Cs[tig] = w1 * (1.f - xv * xv);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if ((tig & 31) == 0) ep4[tig >> 5] = e;
    __syncthreads();
    if (on) {
      if (tig == 0) Ei[a] = (ep4[0] + ep4[1]) + (ep4[2] + ep4[3]) + bw[2 * sp.Nn];
      if (tig < sp.Ndes) {                               // second contraction: thread = descriptor (column of W0)
        const float ev = ns_dot(W0s + tig, ld, Cs, sp.Nn) * qss[tig];
        Ep[(size_t)a * sp.Ndes + tig] = ev;
        Es[tig] = ev;
      }
    }
    __syncthreads();
    if (on && tig < TK)                                  // etil[J][k] = sum_n E'_n cR[t][J][n][k]  (input of the radial force pass)
      etil[(size_t)a * TK + tig] = ns_dot(cRs + (size_t)tig * 16, 1, Es, sp.NR);
    for (int jk = tig + NS_GROUP; on && jk < TK; jk += NS_GROUP) etil[(size_t)a * TK + jk] = ns_dot(cRs + (size_t)jk * 16, 1, Es, sp.NR);
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------
// a6, one launch: p = W0 (s o D), Hc = w1 d2 p, h = s o (Hc W0), gbar = e E' + h  (d1 = 1 - x^2, d2 = -2 x d1, D1.6, C3.8)
// and the parameter-gradient partials of this CTA's atoms (D1.7-D1.17):
//   dL/dW0 = sum A (x) G + Bc (x) sD,  dL/db0 = sum A,  dL/dw1 = sum V,  dL/db1 = sum e,
//   G = s o q, sD = s o D, A = w1 (e d1 + d2 p), Bc = w1 d1, V = e x + d1 p, e = s_e e_struct.
// Same atom ranges as the forward kernel; after a round all threads add the round's rank-2 updates to the CTA's
// W0-gradient accumulator in shared memory (element y = tid + 512 i).  One partial row per CTA, summed in row order by
// k_grad_reduce.
// a7 (radial) rides along: dL/dcR[t][J][n][k] += gbar_n M1[J][k] + E'_n M2[J][k] per atom (cgrad_radial.cuh), the same
// kind of rank-2 update on a [NR][T*KRp] accumulator; its partial row has the layout of k_cgrad_radial's ([n][J][k]),
// one row per CTA (the host points the chunk table of k_grad_reduce at these CTAs).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(NS_THREADS)
k_net_small_bwd(DevSpec sp, SpeciesMap sm, const float *__restrict__ theta, const float *__restrict__ qscale,
                const float *__restrict__ q, const float *__restrict__ D, const float *__restrict__ xbuf,
                const float *__restrict__ Ep, const int *__restrict__ struct_s, const float *__restrict__ e_s,
                const float *__restrict__ scales, const float *__restrict__ M1, const float *__restrict__ M2,
                float *__restrict__ gbar, float *__restrict__ partialW, float *__restrict__ partialB,
                float *__restrict__ partialCR) {
  extern __shared__ __align__(128) float smem[];
  const int ld = sp.ldW, nW = sp.Nn * sp.Ndes, nrow = 2 * sp.Ndes + 3 * sp.Nn, nb = 2 * sp.Nn + 1;
  const int TK = sp.T * sp.KRp, ncr = 2 * sp.NR + 2 * TK, nC = sp.NR * TK;
  const int grp = threadIdx.x >> 7, tig = threadIdx.x & (NS_GROUP - 1);
  float *W0s = smem;                                   // [mu][ld] of this CTA's species
  float *w1s = W0s + (size_t)sp.Nn * ld;               // [Nn]
  float *qss = w1s + sp.Nn;                            // [Ndes]
  float *rows0 = qss + sp.Ndes;                        // per atom: sD | sG | Hc | Av | Bv
  float *accW = rows0 + (size_t)NS_ATOMS * nrow;       // [Nn * Ndes]
  float *red = accW + nW;                              // [atom slot][b0 (Nn) | w1 (Nn) | b1]
  float *crow0 = red + (size_t)NS_ATOMS * nb;          // per atom: gbar[0..NR) | E'[0..NR) | M1[TK] | M2[TK]
  float *accC = crow0 + (size_t)NS_ATOMS * ncr;        // [NR][TK]
  float *crow = crow0 + (size_t)grp * ncr;
  int t, c0, c1;
  ns_range(sm, sp.T, blockIdx.x, t, c0, c1);
  const float *net = theta + sp.offNet + (size_t)t * sp.netSize;
  ns_stage_w0(W0s, net, sp.Nn, sp.Ndes, ld);
  for (int x = threadIdx.x; x < sp.Nn; x += NS_THREADS) w1s[x] = net[nW + sp.Nn + x];
  for (int x = threadIdx.x; x < sp.Ndes; x += NS_THREADS) qss[x] = qscale[x];
  for (int x = threadIdx.x; x < nW; x += NS_THREADS) accW[x] = 0.f;
  for (int x = threadIdx.x; x < nC; x += NS_THREADS) accC[x] = 0.f;
  float *sD = rows0 + (size_t)grp * nrow, *sG = sD + sp.Ndes, *Hc = sG + sp.Ndes, *Av = Hc + sp.Nn, *Bv = Av + sp.Nn;
  const float se = scales[0];
  float accA = 0.f, accV = 0.f, acce = 0.f;            // of neuron tig (of the group's atoms)
  const int mu_first = threadIdx.x / sp.Ndes, nu_first = threadIdx.x - mu_first * sp.Ndes;
  const int dmu = NS_THREADS / sp.Ndes, dnu = NS_THREADS - dmu * sp.Ndes;
  __syncthreads();
  for (int r0 = c0; r0 < c1; r0 += NS_ATOMS) {
    const int a = r0 + grp;
    const bool on = a < c1;
    float e = 0.f, xv = 0.f, epv = 0.f;
    if (on) {
      e = se * e_s[struct_s[a]];
      if (tig < sp.Nn) xv = xbuf[xt_off(a, tig, sp.NnS)];
      if (tig < sp.Ndes) {
        const float s = qss[tig];
        epv = Ep[(size_t)a * sp.Ndes + tig];
        sD[tig] = D[(size_t)a * sp.Ndes + tig] * s;
        sG[tig] = q[(size_t)a * sp.Ndes + tig] * s;
        if (tig < sp.NR) crow[sp.NR + tig] = epv;
      }
      for (int jk = tig; jk < TK; jk += NS_GROUP) { crow[2 * sp.NR + jk] = M1[(size_t)a * TK + jk]; crow[2 * sp.NR + TK + jk] = M2[(size_t)a * TK + jk]; }
      acce += e;
    }
    __syncthreads();
    if (on && tig < sp.Nn) {
      const float p = ns_dot(W0s + (size_t)tig * ld, 1, sD, sp.Ndes), w1 = w1s[tig];
      const float d1 = 1.f - xv * xv, d2 = -2.f * xv * d1;
      const float A = w1 * (e * d1 + d2 * p);
      Hc[tig] = w1 * d2 * p; Av[tig] = A; Bv[tig] = w1 * d1;
      accA += A;
      accV += e * xv + d1 * p;
    }
    __syncthreads();
    if (on && tig < sp.Ndes) {
      const float gb = e * epv + ns_dot(W0s + tig, ld, Hc, sp.Nn) * qss[tig];
      gbar[(size_t)a * sp.Ndes + tig] = gb;
      if (tig < sp.NR) crow[tig] = gb;
    }
    // the round's rank-2 updates to the elements this thread owns
    const int n_on = min(NS_ATOMS, c1 - r0);
    int mu = mu_first, nu = nu_first;
    for (int y = threadIdx.x; y < nW; y += NS_THREADS) {
      float s = accW[y];
#pragma unroll
      for (int w = 0; w < NS_ATOMS; ++w) {
        if (w < n_on) {
          const float *rw = rows0 + (size_t)w * nrow;   // sD | sG | Hc | Av | Bv of atom slot w
          s = fmaf(rw[2 * sp.Ndes + sp.Nn + mu], rw[sp.Ndes + nu], fmaf(rw[2 * sp.Ndes + 2 * sp.Nn + mu], rw[nu], s));
        }
      }
      accW[y] = s;
      mu += dmu; nu += dnu;
      if (nu >= sp.Ndes) { nu -= sp.Ndes; ++mu; }
    }
    __syncthreads();                                     // (the gbar entries of this round are in the rows now)
    for (int y = threadIdx.x; y < nC; y += NS_THREADS) { // a7 radial: element (n, jk)
      const int n = y / TK, jk = y - n * TK;
      float s = accC[y];
#pragma unroll
      for (int w = 0; w < NS_ATOMS; ++w) {
        if (w < n_on) {
          const float *cw = crow0 + (size_t)w * ncr;
          s = fmaf(cw[n], cw[2 * sp.NR + jk], fmaf(cw[sp.NR + n], cw[2 * sp.NR + TK + jk], s));
        }
      }
      accC[y] = s;
    }
    __syncthreads();
  }
  for (int y = threadIdx.x; y < nC; y += NS_THREADS) partialCR[(size_t)blockIdx.x * nC + y] = accC[y];
  for (int y = threadIdx.x; y < nW; y += NS_THREADS) partialW[(size_t)blockIdx.x * nW + y] = accW[y];
  float *rd = red + (size_t)grp * nb;
  if (tig < sp.Nn) { rd[tig] = accA; rd[sp.Nn + tig] = accV; }
  if (tig == 0) rd[2 * sp.Nn] = acce;
  __syncthreads();
  for (int x = threadIdx.x; x < nb; x += NS_THREADS) {
    float s = 0.f;
#pragma unroll
    for (int w = 0; w < NS_ATOMS; ++w) s += red[(size_t)w * nb + x];
    partialB[(size_t)blockIdx.x * nb + x] = s;
  }
}
