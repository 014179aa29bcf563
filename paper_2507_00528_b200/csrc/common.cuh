// common.cuh -- shared device helpers of the GNEP B200 path (fp32 arithmetic, sm_100a).
// Nothing here is shared with oracle/: the oracle is plain C fp64 and is written separately.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define GNEP_MAX_SPECIES_C 4   // == GNEP_MAX_SPECIES of include/gnep.h
#define GNEP_LMAX 8            // largest l_max (paper Eq.7: l = 1..8)
#define GNEP_NLM_MAX 80        // (l,m) slots for l = 1..8; slot lm = l*l - 1 + m, m = 0..2l

// Model constants passed by value to every kernel.
struct DevSpec {
  int T, NR, KR, NA, KA, L, use4, use5, Nn, Ndes, P;
  int nlmS;                   // row stride of the per-atom (l,m) arrays S, T, beta, A1: 24 for l_max <= 4, 84 above
  int NnS;                    // neurons per atom in the hidden-layer buffers x, p: Nn padded to 16 (XT layout, net_tc_kernels.cuh)
  int KRp, KAp;               // basis sizes padded to the template size of the pair kernels
  int offA, offNet, netSize;  // parameter-vector offsets (include/gnep.h layout)
  int ldW;                    // padded shared-memory row stride of W0 (odd -> conflict-free)
  int loss_mode;
  float rcRinv, rcAinv;
  float lam_e, lam_f, lam_v, lam_2;
};

// l of slot lm
__host__ __device__ constexpr int blm_l(int lm) {
  int l = 1;
  while ((l + 1) * (l + 1) - 1 <= lm) ++l;
  return l;
}

// 2*C_lm with C_lm = (2l+1)/(4 pi) * Chat_lm (R11-R12): Chat_lm is fixed by the addition theorem
// sum_m Chat_lm b_lm(r1) b_lm(r2) = r1^l r2^l P_l(cos theta12) for the paper's b_lm (App.B); one entry for m = 0, then one
// per (cos, sin) pair.  Compile-time table: the same for every model, so nothing per-handle lives in constant memory.
#define GNEP_C2(l, chat) ((float)(2.0 * (2 * (l) + 1) / (4.0 * 3.14159265358979323846) * (chat)))
#define GNEP_C2P(l, chat) GNEP_C2(l, chat), GNEP_C2(l, chat)
__constant__ float c_C2[GNEP_NLM_MAX + 4] = {
    GNEP_C2(1, 1.0), GNEP_C2P(1, 1.0),
    GNEP_C2(2, 1.0 / 4), GNEP_C2P(2, 3.0), GNEP_C2P(2, 3.0 / 4),
    GNEP_C2(3, 1.0 / 4), GNEP_C2P(3, 3.0 / 8), GNEP_C2P(3, 15.0 / 4), GNEP_C2P(3, 5.0 / 8),
    GNEP_C2(4, 1.0 / 64), GNEP_C2P(4, 5.0 / 8), GNEP_C2P(4, 5.0 / 16), GNEP_C2P(4, 35.0 / 8), GNEP_C2P(4, 35.0 / 64),
    GNEP_C2(5, 1.0 / 64), GNEP_C2P(5, 15.0 / 64), GNEP_C2P(5, 105.0 / 16), GNEP_C2P(5, 35.0 / 128), GNEP_C2P(5, 315.0 / 64),
    GNEP_C2P(5, 63.0 / 128),
    GNEP_C2(6, 1.0 / 256), GNEP_C2P(6, 21.0 / 64), GNEP_C2P(6, 105.0 / 512), GNEP_C2P(6, 105.0 / 128), GNEP_C2P(6, 63.0 / 256),
    GNEP_C2P(6, 693.0 / 128), GNEP_C2P(6, 231.0 / 512),
    GNEP_C2(7, 1.0 / 256), GNEP_C2P(7, 7.0 / 1024), GNEP_C2P(7, 21.0 / 512), GNEP_C2P(7, 21.0 / 1024), GNEP_C2P(7, 231.0 / 256),
    GNEP_C2P(7, 231.0 / 1024), GNEP_C2P(7, 3003.0 / 512), GNEP_C2P(7, 429.0 / 1024),
    GNEP_C2(8, 1.0 / 16384), GNEP_C2P(8, 9.0 / 1024), GNEP_C2P(8, 315.0 / 2048), GNEP_C2P(8, 1155.0 / 1024),
    GNEP_C2P(8, 693.0 / 4096), GNEP_C2P(8, 9009.0 / 1024), GNEP_C2P(8, 429.0 / 2048), GNEP_C2P(8, 6435.0 / 1024),
    GNEP_C2P(8, 6435.0 / 16384),
    0.f, 0.f, 0.f, 0.f};
// kappa4 = -5 sqrt(14) / (448 pi^(3/2)) (R14); kappa5 = 3 / (16 pi^2) (R41)
#define GNEP_KAPPA4 (-0.0074994808266641f)
#define GNEP_KAPPA5 (0.018997721932938f)

// ---------------------------------------------------------------------------------------------
// Pair geometry: d = |r| and 1/d from one MUFU.RSQ and one Newton step (relative error ~1e-7, as sqrtf + division).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void pair_len(float d2, float &d, float &rinv) {
  const float y = rsqrtf(d2);
  const float e = fmaf(-d2 * y, y, 1.f);
  rinv = fmaf(0.5f * y, e, y);
  d = d2 * rinv;
}

// ---------------------------------------------------------------------------------------------
// Chebyshev radial basis (paper Eq.6, App.A):  f_k = 1/2 (T_k(xi)+1) f_c,  xi = 2 (d/rc - 1)^2 - 1,
// f_c = 1/2 (1 + cos(pi d/rc)); d/rc is clamped at 1, where f_k = f_k' = 0 exactly
// (real pairs have d < rc; the padding dummies of the angular list sit at 2 rc).
// cheb_T / cheb_TD give the pieces, so that sums over pairs can be accumulated per Chebyshev term:
//   f_0 = 2 hfc,  f_k = hfc T_k + hfc;   f_0' = 2 hfcp,  f_k' = D_k hdf + T_k hfcp + hfcp   (D_k = dT_k/dxi)
// ---------------------------------------------------------------------------------------------
#define GNEP_PI_F 3.14159265358979f
// sin(pi t), cos(pi t) for t in [0, 1] from the Taylor polynomials about t = 1/2 (x = pi (t - 1/2), |x| <= pi/2):
// cos(pi t) = -sin x, sin(pi t) = cos x; truncation 6e-8 / 7e-9 absolute, i.e. fp32 rounding level, in ~16 instructions
// (sincospif spends about twice that on its general range reduction).
__device__ __forceinline__ float cospi01(float t) {
  const float x = GNEP_PI_F * (t - 0.5f), x2 = x * x;
  float p = fmaf(x2, -2.5052108e-8f, 2.7557319e-6f);
  p = fmaf(x2, p, -1.9841270e-4f);
  p = fmaf(x2, p, 8.3333333e-3f);
  p = fmaf(x2, p, -1.6666667e-1f);
  return -fmaf(x * x2, p, x);
}
__device__ __forceinline__ void sincospi01(float t, float &sn, float &cs) {
  const float x = GNEP_PI_F * (t - 0.5f), x2 = x * x;
  float p = fmaf(x2, -2.5052108e-8f, 2.7557319e-6f);
  p = fmaf(x2, p, -1.9841270e-4f);
  p = fmaf(x2, p, 8.3333333e-3f);
  p = fmaf(x2, p, -1.6666667e-1f);
  cs = -fmaf(x * x2, p, x);
  float c = fmaf(x2, 2.0876757e-9f, -2.7557319e-7f);
  c = fmaf(x2, c, 2.4801587e-5f);
  c = fmaf(x2, c, -1.3888889e-3f);
  c = fmaf(x2, c, 4.1666667e-2f);
  c = fmaf(x2, c, -0.5f);
  sn = fmaf(x2, c, 1.f);
}
template <int KT>
__device__ __forceinline__ void cheb_T(float d, float rcinv, float (&Tk)[KT], float &hfc) {
  const float t = fminf(d * rcinv, 1.f);
  const float x = t - 1.f;
  const float xi = 2.f * x * x - 1.f;
  hfc = t < 1.f ? 0.25f * (1.f + cospi01(t)) : 0.f;                 // 1/2 f_c
  Tk[0] = 1.f;
  if (KT > 1) Tk[1] = xi;
#pragma unroll
  for (int k = 2; k < KT; ++k) Tk[k] = 2.f * xi * Tk[k - 1] - Tk[k - 2];
}
template <int KT>
__device__ __forceinline__ void cheb_TD(float d, float rcinv, float (&Tk)[KT], float (&Dk)[KT], float &hfc, float &hfcp,
                                        float &hdf) {
  const float t = fminf(d * rcinv, 1.f);
  const float x = t - 1.f;
  const float xi = 2.f * x * x - 1.f;
  float sn, cs;
  sincospi01(t, sn, cs);
  const bool in = t < 1.f;
  hfc = in ? 0.25f * (1.f + cs) : 0.f;                              // 1/2 f_c
  hfcp = in ? -0.25f * GNEP_PI_F * rcinv * sn : 0.f;                // 1/2 f_c'
  hdf = hfc * 4.f * x * rcinv;                                      // 1/2 f_c dxi/dd
  Tk[0] = 1.f; Dk[0] = 0.f;
  if (KT > 1) { Tk[1] = xi; Dk[1] = 1.f; }
#pragma unroll
  for (int k = 2; k < KT; ++k) {
    Tk[k] = 2.f * xi * Tk[k - 1] - Tk[k - 2];
    Dk[k] = 2.f * Tk[k - 1] + 2.f * xi * Dk[k - 1] - Dk[k - 2];
  }
}

template <int KT>
__device__ __forceinline__ void cheb_f(float d, float rcinv, float (&f)[KT]) {
  float Tk[KT], hfc;
  cheb_T<KT>(d, rcinv, Tk, hfc);
  f[0] = 2.f * hfc;
#pragma unroll
  for (int k = 1; k < KT; ++k) f[k] = fmaf(hfc, Tk[k], hfc);
}

template <int KT>
__device__ __forceinline__ void cheb_ffp(float d, float rcinv, float (&f)[KT], float (&fp)[KT]) {
  float Tk[KT], Dk[KT], hfc, hfcp, hdf;
  cheb_TD<KT>(d, rcinv, Tk, Dk, hfc, hfcp, hdf);
  f[0] = 2.f * hfc; fp[0] = 2.f * hfcp;
#pragma unroll
  for (int k = 1; k < KT; ++k) {
    f[k] = fmaf(hfc, Tk[k], hfc);
    fp[k] = fmaf(Dk[k], hdf, fmaf(Tk[k], hfcp, hfcp));
  }
}

// (f_k, f_k') as register pairs, built with packed FP32 FMAs (sm_100 FFMA2: two fp32 FMAs per issue slot): the pair
// (T_k, D_k) runs through one recurrence, (T_k, D_k) = 2 xi (T_k-1, D_k-1) - (T_k-2, D_k-2) + (0, 2 T_k-1), and
// (f_k, f_k') = (hfc, hdf) (T_k, D_k) + (hfc, hfcp (T_k + 1)).  Same values as cheb_ffp up to rounding order.
template <int KT>
__device__ __forceinline__ void cheb_ffp2(float d, float rcinv, float2 (&ffp)[KT]) {
  const float t = fminf(d * rcinv, 1.f);
  const float x = t - 1.f;
  const float xi = 2.f * x * x - 1.f;
  float sn, cs;
  sincospi01(t, sn, cs);
  const bool in = t < 1.f;
  const float hfc = in ? 0.25f * (1.f + cs) : 0.f;
  const float hfcp = in ? -0.25f * GNEP_PI_F * rcinv * sn : 0.f;
  const float hdf = hfc * 4.f * x * rcinv;
  const float2 sc = make_float2(hfc, hdf), xx = make_float2(2.f * xi, 2.f * xi);
  auto combine = [&](const float2 &td) { return __ffma2_rn(sc, td, make_float2(hfc, fmaf(hfcp, td.x, hfcp))); };
  float2 p2 = make_float2(1.f, 0.f), p1 = make_float2(xi, 1.f);
  ffp[0] = make_float2(2.f * hfc, 2.f * hfcp);
  if (KT > 1) ffp[1] = combine(p1);
#pragma unroll
  for (int k = 2; k < KT; ++k) {
    float2 c = __ffma2_rn(xx, p1, make_float2(-p2.x, -p2.y));
    c.y = fmaf(2.f, p1.x, c.y);
    ffp[k] = combine(c);
    p2 = p1; p1 = c;
  }
}

// ---------------------------------------------------------------------------------------------
// Real harmonics of a UNIT vector (paper App.B): emits, for each of the LMAX (LMAX + 2) (l,m) slots,
// b = b_lm(rhat) and g = (grad b_lm)(rhat)  [polynomial gradient, r^2 terms differentiated, then r=1].
// With B_lm = b_lm(r)/d^l:  B_lm = b,  grad B_lm = (g - l b rhat) / d.
// F is called as f(lm, l, b, gx, gy, gz) with literal lm so that register arrays index statically.
// ---------------------------------------------------------------------------------------------
template <int LMAX, class F>
__device__ __forceinline__ void blm_unit(float x, float y, float z, F f) {
  static_assert(LMAX == 4 || LMAX == 8, "harmonics are instantiated for l_max 4 and 8");
  float x2 = x * x, y2 = y * y, z2 = z * z;
  float xy = x * y, xz = x * z, yz = y * z;
  float d2 = x2 - y2;
  // l = 1
  f(0, 1, z, 0.f, 0.f, 1.f);
  f(1, 1, x, 1.f, 0.f, 0.f);
  f(2, 1, y, 0.f, 1.f, 0.f);
  // l = 2
  f(3, 2, 3.f * z2 - 1.f, -2.f * x, -2.f * y, 4.f * z);
  f(4, 2, xz, z, 0.f, x);
  f(5, 2, yz, 0.f, z, y);
  f(6, 2, d2, 2.f * x, -2.f * y, 0.f);
  f(7, 2, 2.f * xy, 2.f * y, 2.f * x, 0.f);
  // l = 3
  float a5 = 5.f * z2 - 1.f;
  f(8, 3, (5.f * z2 - 3.f) * z, -6.f * xz, -6.f * yz, 9.f * z2 - 3.f);
  f(9, 3, a5 * x, a5 - 2.f * x2, -2.f * xy, 8.f * xz);
  f(10, 3, a5 * y, -2.f * xy, a5 - 2.f * y2, 8.f * yz);
  f(11, 3, d2 * z, 2.f * xz, -2.f * yz, d2);
  f(12, 3, 2.f * xy * z, 2.f * yz, 2.f * xz, 2.f * xy);
  f(13, 3, (x2 - 3.f * y2) * x, 3.f * d2, -6.f * xy, 0.f);
  f(14, 3, (3.f * x2 - y2) * y, 6.f * xy, 3.f * d2, 0.f);
  // l = 4
  float p = (7.f * z2 - 3.f) * z;
  float w = 7.f * z2 - 1.f;
  float c3 = 15.f * z2 - 3.f;
  float cx = (x2 - 3.f * y2) * x, cy = (3.f * x2 - y2) * y;
  f(15, 4, (35.f * z2 - 30.f) * z2 + 3.f, (12.f - 60.f * z2) * x, (12.f - 60.f * z2) * y, (80.f * z2 - 48.f) * z);
  f(16, 4, p * x, p - 6.f * z * x2, -6.f * z * xy, c3 * x);
  f(17, 4, p * y, -6.f * z * xy, p - 6.f * z * y2, c3 * y);
  f(18, 4, w * d2, 2.f * x * (w - d2), -2.f * y * (w + d2), 12.f * z * d2);
  f(19, 4, 2.f * w * xy, 2.f * y * (w - 2.f * x2), 2.f * x * (w - 2.f * y2), 24.f * xy * z);
  f(20, 4, cx * z, 3.f * d2 * z, -6.f * xy * z, cx);
  f(21, 4, cy * z, 6.f * xy * z, 3.f * d2 * z, cy);
  f(22, 4, x2 * x2 - 6.f * x2 * y2 + y2 * y2, 4.f * cx, -4.f * cy, 0.f);
  f(23, 4, 4.f * xy * d2, 4.f * cy, 4.f * cx, 0.f);
  if constexpr (LMAX > 4) {
    // l = 5..8 (Eq.B5.1-B8.17): b_lm = Z_lm'(z, r^2) * Re/Im (x + i y)^m', m' = 0 for m = 0 and m' = ceil(m/2)
    // otherwise.  With cm = Re (x+iy)^m', sm = Im (x+iy)^m' and, at r = 1, Z, Zz = dZ/dz, Zr = dZ/d(r^2):
    //   grad (Z cm) = Z m' (c_{m'-1}, -s_{m'-1}, 0) + cm (2 Zr x, 2 Zr y, Zz + 2 Zr z)      (polynomial gradient)
    //   grad (Z sm) = Z m' (s_{m'-1},  c_{m'-1}, 0) + sm (2 Zr x, 2 Zr y, Zz + 2 Zr z)
    float cm[9], sm[9];
    cm[0] = 1.f; sm[0] = 0.f;
#pragma unroll
    for (int m = 1; m <= 8; ++m) { cm[m] = x * cm[m - 1] - y * sm[m - 1]; sm[m] = x * sm[m - 1] + y * cm[m - 1]; }
    const float z3 = z2 * z, z4 = z2 * z2, z5 = z4 * z, z6 = z4 * z2, z7 = z6 * z, z8 = z4 * z4;
    auto zero = [&](int lm, int l, float Z, float Zz, float Zr) { f(lm, l, Z, 2.f * Zr * x, 2.f * Zr * y, Zz + 2.f * Zr * z); };
    auto pair = [&](int lm, int l, int m, float Z, float Zz, float Zr) {
      const float fm = (float)m, w = Zz + 2.f * Zr * z, zx = 2.f * Zr * x, zy = 2.f * Zr * y;
      f(lm, l, Z * cm[m], Z * fm * cm[m - 1] + zx * cm[m], -Z * fm * sm[m - 1] + zy * cm[m], w * cm[m]);
      f(lm + 1, l, Z * sm[m], Z * fm * sm[m - 1] + zx * sm[m], Z * fm * cm[m - 1] + zy * sm[m], w * sm[m]);
    };
    // l = 5, slots 24..34
    zero(24, 5, 63.f * z5 - 70.f * z3 + 15.f * z, 315.f * z4 - 210.f * z2 + 15.f, -70.f * z3 + 30.f * z);
    pair(25, 5, 1, 21.f * z4 - 14.f * z2 + 1.f, 84.f * z3 - 28.f * z, -14.f * z2 + 2.f);
    pair(27, 5, 2, 3.f * z3 - z, 9.f * z2 - 1.f, -z);
    pair(29, 5, 3, 9.f * z2 - 1.f, 18.f * z, -1.f);
    pair(31, 5, 4, z, 1.f, 0.f);
    pair(33, 5, 5, 1.f, 0.f, 0.f);
    // l = 6, slots 35..47
    zero(35, 6, 231.f * z6 - 315.f * z4 + 105.f * z2 - 5.f, 1386.f * z5 - 1260.f * z3 + 210.f * z, -315.f * z4 + 210.f * z2 - 15.f);
    pair(36, 6, 1, 33.f * z5 - 30.f * z3 + 5.f * z, 165.f * z4 - 90.f * z2 + 5.f, -30.f * z3 + 10.f * z);
    pair(38, 6, 2, 33.f * z4 - 18.f * z2 + 1.f, 132.f * z3 - 36.f * z, -18.f * z2 + 2.f);
    pair(40, 6, 3, 11.f * z3 - 3.f * z, 33.f * z2 - 3.f, -3.f * z);
    pair(42, 6, 4, 11.f * z2 - 1.f, 22.f * z, -1.f);
    pair(44, 6, 5, z, 1.f, 0.f);
    pair(46, 6, 6, 1.f, 0.f, 0.f);
    // l = 7, slots 48..62
    zero(48, 7, 429.f * z7 - 693.f * z5 + 315.f * z3 - 35.f * z, 3003.f * z6 - 3465.f * z4 + 945.f * z2 - 35.f,
         -693.f * z5 + 630.f * z3 - 105.f * z);
    pair(49, 7, 1, 429.f * z6 - 495.f * z4 + 135.f * z2 - 5.f, 2574.f * z5 - 1980.f * z3 + 270.f * z, -495.f * z4 + 270.f * z2 - 15.f);
    pair(51, 7, 2, 143.f * z5 - 110.f * z3 + 15.f * z, 715.f * z4 - 330.f * z2 + 15.f, -110.f * z3 + 30.f * z);
    pair(53, 7, 3, 143.f * z4 - 66.f * z2 + 3.f, 572.f * z3 - 132.f * z, -66.f * z2 + 6.f);
    pair(55, 7, 4, 13.f * z3 - 3.f * z, 39.f * z2 - 3.f, -3.f * z);
    pair(57, 7, 5, 13.f * z2 - 1.f, 26.f * z, -1.f);
    pair(59, 7, 6, z, 1.f, 0.f);
    pair(61, 7, 7, 1.f, 0.f, 0.f);
    // l = 8, slots 63..79
    zero(63, 8, 6435.f * z8 - 12012.f * z6 + 6930.f * z4 - 1260.f * z2 + 35.f, 51480.f * z7 - 72072.f * z5 + 27720.f * z3 - 2520.f * z,
         -12012.f * z6 + 13860.f * z4 - 3780.f * z2 + 140.f);
    pair(64, 8, 1, 715.f * z7 - 1001.f * z5 + 385.f * z3 - 35.f * z, 5005.f * z6 - 5005.f * z4 + 1155.f * z2 - 35.f,
         -1001.f * z5 + 770.f * z3 - 105.f * z);
    pair(66, 8, 2, 143.f * z6 - 143.f * z4 + 33.f * z2 - 1.f, 858.f * z5 - 572.f * z3 + 66.f * z, -143.f * z4 + 66.f * z2 - 3.f);
    pair(68, 8, 3, 39.f * z5 - 26.f * z3 + 3.f * z, 195.f * z4 - 78.f * z2 + 3.f, -26.f * z3 + 6.f * z);
    pair(70, 8, 4, 65.f * z4 - 26.f * z2 + 1.f, 260.f * z3 - 52.f * z, -26.f * z2 + 2.f);
    pair(72, 8, 5, 5.f * z3 - z, 15.f * z2 - 1.f, -z);
    pair(74, 8, 6, 15.f * z2 - 1.f, 30.f * z, -1.f);
    pair(76, 8, 7, z, 1.f, 0.f);
    pair(78, 8, 8, 1.f, 0.f, 0.f);
  }
}

// 4-body cubic invariant of the l=2 moments s[0..4] (R14): P4, gradient, Hessian*t
__device__ __forceinline__ float p4_value(const float *s) {
  float s0 = s[0], s1 = s[1], s2 = s[2], s3 = s[3], s4 = s[4];
  return s0 * s0 * s0 + 18.f * s0 * (s1 * s1 + s2 * s2) - 9.f * s0 * (s3 * s3 + s4 * s4) +
         54.f * s3 * (s1 * s1 - s2 * s2) + 108.f * s1 * s2 * s4;
}
__device__ __forceinline__ void p4_grad(const float *s, float *g) {
  float s0 = s[0], s1 = s[1], s2 = s[2], s3 = s[3], s4 = s[4];
  g[0] = 3.f * s0 * s0 + 18.f * (s1 * s1 + s2 * s2) - 9.f * (s3 * s3 + s4 * s4);
  g[1] = 36.f * s0 * s1 + 108.f * s3 * s1 + 108.f * s2 * s4;
  g[2] = 36.f * s0 * s2 - 108.f * s3 * s2 + 108.f * s1 * s4;
  g[3] = -18.f * s0 * s3 + 54.f * (s1 * s1 - s2 * s2);
  g[4] = -18.f * s0 * s4 + 108.f * s1 * s2;
}
__device__ __forceinline__ void p4_hess_vec(const float *s, const float *t, float *h) {
  float s0 = s[0], s1 = s[1], s2 = s[2], s3 = s[3], s4 = s[4];
  h[0] = 6.f * s0 * t[0] + 36.f * s1 * t[1] + 36.f * s2 * t[2] - 18.f * s3 * t[3] - 18.f * s4 * t[4];
  h[1] = 36.f * s1 * t[0] + (36.f * s0 + 108.f * s3) * t[1] + 108.f * s4 * t[2] + 108.f * s1 * t[3] + 108.f * s2 * t[4];
  h[2] = 36.f * s2 * t[0] + 108.f * s4 * t[1] + (36.f * s0 - 108.f * s3) * t[2] - 108.f * s2 * t[3] + 108.f * s1 * t[4];
  h[3] = -18.f * s3 * t[0] + 108.f * s1 * t[1] - 108.f * s2 * t[2] - 18.f * s0 * t[3];
  h[4] = -18.f * s4 * t[0] + 108.f * s2 * t[1] + 108.f * s1 * t[2] - 18.f * s0 * t[4];
}

// 5-body quartic invariant of the l=1 moments s[0..2] (R41): q5 = kappa5 |s|^4; value, gradient, Hessian*t
__device__ __forceinline__ float p5_value(const float *s) {
  const float n2 = s[0] * s[0] + s[1] * s[1] + s[2] * s[2];
  return GNEP_KAPPA5 * n2 * n2;
}
__device__ __forceinline__ void p5_grad(const float *s, float *g) {
  const float c = 4.f * GNEP_KAPPA5 * (s[0] * s[0] + s[1] * s[1] + s[2] * s[2]);
  g[0] = c * s[0]; g[1] = c * s[1]; g[2] = c * s[2];
}
__device__ __forceinline__ void p5_hess_vec(const float *s, const float *t, float *h) {
  const float n2 = s[0] * s[0] + s[1] * s[1] + s[2] * s[2], st = s[0] * t[0] + s[1] * t[1] + s[2] * t[2];
  const float a = 4.f * GNEP_KAPPA5 * n2, b = 8.f * GNEP_KAPPA5 * st;
  h[0] = a * t[0] + b * s[0]; h[1] = a * t[1] + b * s[1]; h[2] = a * t[2] + b * s[2];
}

// 8 consecutive floats at a 32-byte aligned address as ONE 256-bit access (sm_100: LDG/STG.256): half as many requests
// as two 128-bit ones, which is what row-per-thread / row-per-lane patterns pay for (a different line per lane)
struct float8 { float4 lo, hi; };
__device__ __forceinline__ float8 ldg256(const float *p) {
  float8 r;
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(r.lo.x), "=f"(r.lo.y), "=f"(r.lo.z), "=f"(r.lo.w), "=f"(r.hi.x), "=f"(r.hi.y), "=f"(r.hi.z), "=f"(r.hi.w)
               : "l"(p));
  return r;
}
// the same for data that is streamed once (pair lists): no L1 allocation, so that the lines of the per-atom rows the
// sweep gathers (etil_j, u_j) stay resident in L1
__device__ __forceinline__ float8 ldg256_stream(const float *p) {
  float8 r;
  asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(r.lo.x), "=f"(r.lo.y), "=f"(r.lo.z), "=f"(r.lo.w), "=f"(r.hi.x), "=f"(r.hi.y), "=f"(r.hi.z), "=f"(r.hi.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void stg256(float *p, const float4 &a, const float4 &b) {
  asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(a.x), "f"(a.y), "f"(a.z), "f"(a.w), "f"(b.x),
               "f"(b.y), "f"(b.z), "f"(b.w)
               : "memory");
}
// stage the expansion coefficients c[I][J][n][k] into shared memory with k padded to KT (zeros)
__device__ __forceinline__ void stage_coeff(float *dst, const float *src, int rows, int K, int KT) {
  for (int x = threadIdx.x; x < rows * KT; x += blockDim.x) {
    int r = x / KT, k = x - r * KT;
    dst[x] = (k < K) ? src[r * K + k] : 0.f;
  }
}
