// neighbor.cuh -- periodic cell-list neighbour builder (paper Eq.2; R7-R9, row a0).
// Runs once per loaded batch.  The distance test is fp64 with explicit round-to-nearest intrinsics
// (no FMA contraction) in a fixed operation order, so that the result is bit-identical to a plain
// IEEE evaluation of   t = (sa*a + sb*b) + sc*c ; d = (r_j - r_i) + t ; d2 = (dx*dx + dy*dy) + dz*dz.
#pragma once
#include "common.cuh"

struct StructGeo {
  double cell[9];   // rows a, b, c
  double inv[9];    // u_a = pos . inv[0..2], u_b = pos . inv[3..5], u_c = pos . inv[6..8]
  int nb[3];        // bins per axis (fractional width 1/nb >= rc/h, or 1 bin)
  int m[3];         // bins to search on each side
  int bin_base;     // first global bin of this structure
  int a0, a1;       // atom range (input order)
};

__device__ __forceinline__ double lattice_comb(double sa, double sb, double sc, double a, double b, double c) {
  return __dadd_rn(__dadd_rn(__dmul_rn(sa, a), __dmul_rn(sb, b)), __dmul_rn(sc, c));
}

// one thread per atom: move into the cell by whole lattice vectors, compute its bin, count the bin
__global__ void k_wrap_bin(int N, const int *__restrict__ struct_of, const StructGeo *__restrict__ geo,
                           const double *__restrict__ pos_in, double *__restrict__ wpos,
                           int *__restrict__ binid, int *__restrict__ bin_count) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const StructGeo &g = geo[struct_of[i]];
  double x = pos_in[3 * i], y = pos_in[3 * i + 1], z = pos_in[3 * i + 2];
  double u[3], fl[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    u[a] = __dadd_rn(__dadd_rn(__dmul_rn(x, g.inv[3 * a]), __dmul_rn(y, g.inv[3 * a + 1])), __dmul_rn(z, g.inv[3 * a + 2]));
    fl[a] = floor(u[a]);
  }
  if (fl[0] != 0.0 || fl[1] != 0.0 || fl[2] != 0.0) {
    x = __dsub_rn(x, lattice_comb(fl[0], fl[1], fl[2], g.cell[0], g.cell[3], g.cell[6]));
    y = __dsub_rn(y, lattice_comb(fl[0], fl[1], fl[2], g.cell[1], g.cell[4], g.cell[7]));
    z = __dsub_rn(z, lattice_comb(fl[0], fl[1], fl[2], g.cell[2], g.cell[5], g.cell[8]));
  }
  wpos[3 * i] = x; wpos[3 * i + 1] = y; wpos[3 * i + 2] = z;
  int b[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    int v = (int)((u[a] - fl[a]) * g.nb[a]);
    b[a] = min(max(v, 0), g.nb[a] - 1);
  }
  int bin = g.bin_base + (b[0] * g.nb[1] + b[1]) * g.nb[2] + b[2];
  binid[i] = bin;
  atomicAdd(&bin_count[bin], 1);
}

__global__ void k_bin_fill(int N, const int *__restrict__ binid, const int *__restrict__ bin_start,
                           int *__restrict__ bin_cursor, int *__restrict__ bin_atoms) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  int b = binid[i];
  int slot = atomicAdd(&bin_cursor[b], 1);
  bin_atoms[bin_start[b] + slot] = i;
}

__device__ __forceinline__ int floor_div(int a, int b) { int q = a / b; return (a % b != 0 && ((a < 0) != (b < 0))) ? q - 1 : q; }

// Visit every (j, shift) candidate of atom i through the extended-bin stencil; F(j, sa, sb, sc, dx, dy, dz, d2)
template <class F>
__device__ __forceinline__ void visit_candidates(int i, const StructGeo &g, const double *__restrict__ wpos,
                                                 const int *__restrict__ binid, const int *__restrict__ bin_start,
                                                 const int *__restrict__ bin_atoms, F f) {
  double xi = wpos[3 * i], yi = wpos[3 * i + 1], zi = wpos[3 * i + 2];
  int lb = binid[i] - g.bin_base;
  int bc = lb % g.nb[2], bb = (lb / g.nb[2]) % g.nb[1], ba = lb / (g.nb[2] * g.nb[1]);
  for (int da = -g.m[0]; da <= g.m[0]; ++da) {
    int ea = ba + da, sa = floor_div(ea, g.nb[0]), ca = ea - sa * g.nb[0];
    for (int db = -g.m[1]; db <= g.m[1]; ++db) {
      int eb = bb + db, sb = floor_div(eb, g.nb[1]), cb = eb - sb * g.nb[1];
      for (int dc = -g.m[2]; dc <= g.m[2]; ++dc) {
        int ec = bc + dc, sc = floor_div(ec, g.nb[2]), cc = ec - sc * g.nb[2];
        double tx = lattice_comb((double)sa, (double)sb, (double)sc, g.cell[0], g.cell[3], g.cell[6]);
        double ty = lattice_comb((double)sa, (double)sb, (double)sc, g.cell[1], g.cell[4], g.cell[7]);
        double tz = lattice_comb((double)sa, (double)sb, (double)sc, g.cell[2], g.cell[5], g.cell[8]);
        int bin = g.bin_base + (ca * g.nb[1] + cb) * g.nb[2] + cc;
        int e0 = bin_start[bin], e1 = bin_start[bin + 1];
        for (int e = e0; e < e1; ++e) {
          int j = bin_atoms[e];
          if (j == i && sa == 0 && sb == 0 && sc == 0) continue;
          double dx = __dadd_rn(__dsub_rn(wpos[3 * j], xi), tx);
          double dy = __dadd_rn(__dsub_rn(wpos[3 * j + 1], yi), ty);
          double dz = __dadd_rn(__dsub_rn(wpos[3 * j + 2], zi), tz);
          double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
          f(j, sa, sb, sc, dx, dy, dz, d2);
        }
      }
    }
  }
}

__global__ void k_nbr_count(int N, const int *__restrict__ struct_of, const StructGeo *__restrict__ geo,
                            const double *__restrict__ wpos, const int *__restrict__ binid,
                            const int *__restrict__ bin_start, const int *__restrict__ bin_atoms,
                            double rcR2, double rcA2, int *__restrict__ cntR, int *__restrict__ cntA) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  int nR = 0, nA = 0;
  visit_candidates(i, geo[struct_of[i]], wpos, binid, bin_start, bin_atoms,
                   [&](int, int, int, int, double, double, double, double d2) {
                     if (d2 < rcR2) { ++nR; if (d2 < rcA2) ++nA; }
                   });
  cntR[i] = nR; cntA[i] = nA;
}

// sort key of a pair inside its row: (j local to the structure, sa, sb, sc) ascending
__device__ __forceinline__ unsigned long long pair_key(int jl, int sa, int sb, int sc) {
  return ((unsigned long long)(unsigned)jl << 24) | ((unsigned long long)(sa + 128) << 16) |
         ((unsigned long long)(sb + 128) << 8) | (unsigned long long)(sc + 128);
}
#define KEY_ANG_BIT (1ull << 62)     // set on pairs that are also in the angular list

__global__ void k_nbr_fill(int N, const int *__restrict__ struct_of, const StructGeo *__restrict__ geo,
                           const double *__restrict__ wpos, const int *__restrict__ binid,
                           const int *__restrict__ bin_start, const int *__restrict__ bin_atoms,
                           double rcR2, double rcA2, const int64_t *__restrict__ rowR,
                           unsigned long long *__restrict__ ekey, float *__restrict__ er) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const StructGeo &g = geo[struct_of[i]];
  int64_t p = rowR[i];
  int a0 = g.a0;
  visit_candidates(i, g, wpos, binid, bin_start, bin_atoms,
                   [&](int j, int sa, int sb, int sc, double dx, double dy, double dz, double d2) {
                     if (d2 < rcR2) {
                       unsigned long long k = pair_key(j - a0, sa, sb, sc);
                       if (d2 < rcA2) k |= KEY_ANG_BIT;
                       ekey[p] = k;
                       er[3 * p] = (float)dx; er[3 * p + 1] = (float)dy; er[3 * p + 2] = (float)dz;
                       ++p;
                     }
                   });
}

// One warp per atom (input order i).  Ranks every entry of the row (O(M^2/32) per lane) and scatters it to
//   - the canonical export lists (input atom order, ascending (j, shift))                     [parity aid]
//   - the internal lists (atoms sorted by species; rows ordered by neighbour species J, then canonically)
// pair record = float4(r_ij.x, r_ij.y, r_ij.z, bits(internal index of j)).
__global__ void k_nbr_scatter(int N, int T, const int *__restrict__ struct_of, const StructGeo *__restrict__ geo,
                              const int *__restrict__ type, const int *__restrict__ inv_perm,
                              const int64_t *__restrict__ rowR, const int64_t *__restrict__ rowA,
                              const int *__restrict__ rowRs, const int *__restrict__ rowAs,
                              const unsigned long long *__restrict__ ekey, const float *__restrict__ er,
                              int *__restrict__ expR_j, int *__restrict__ expR_sh, int *__restrict__ expA_j,
                              int *__restrict__ expA_sh, float4 *__restrict__ pairR, float4 *__restrict__ pairA,
                              int *__restrict__ shA, int *__restrict__ segR, int *__restrict__ segA,
                              int *__restrict__ atomA) {
  int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (i >= N) return;
  int a0 = geo[struct_of[i]].a0;
  int64_t r0 = rowR[i], r1 = rowR[i + 1];
  int a = inv_perm[i];
  int baseRs = rowRs[a], baseAs = rowAs[a];
  int64_t baseA = rowA[i];
  const unsigned long long KM = KEY_ANG_BIT - 1;
  int cntJ[4] = {0, 0, 0, 0}, cntJA[4] = {0, 0, 0, 0};   // GNEP_MAX_SPECIES
  for (int64_t e = r0 + lane; e < r1; e += 32) {
    unsigned long long ke = ekey[e];
    bool ang = (ke & KEY_ANG_BIT) != 0;
    unsigned long long kc = ke & KM;
    int j = a0 + (int)(kc >> 24);
    int J = type[j];
    unsigned long long ki = ((unsigned long long)J << 56) | kc;
    int rankC = 0, rankCA = 0, rankI = 0, rankIA = 0;
    for (int64_t o = r0; o < r1; ++o) {
      unsigned long long ko = ekey[o];
      bool oang = (ko & KEY_ANG_BIT) != 0;
      unsigned long long kco = ko & KM;
      int Jo = type[a0 + (int)(kco >> 24)];
      unsigned long long kio = ((unsigned long long)Jo << 56) | kco;
      bool lessC = kco < kc, lessI = kio < ki;
      rankC += lessC; rankI += lessI;
      if (oang) { rankCA += lessC; rankIA += lessI; }
    }
    int sh = (int)(kc & 0xffffffull);
    expR_j[r0 + rankC] = j; expR_sh[r0 + rankC] = sh;
    float4 rec = make_float4(er[3 * e], er[3 * e + 1], er[3 * e + 2], __int_as_float(inv_perm[j]));
    pairR[baseRs + rankI] = rec;
    if (ang) {
      expA_j[baseA + rankCA] = j; expA_sh[baseA + rankCA] = sh;
      pairA[baseAs + rankIA] = rec;
      shA[baseAs + rankIA] = sh;
      atomA[baseAs + rankIA] = a | (J << 28) | (type[i] << 30);   // central atom, neighbour species, central species
      cntJA[J] += 1;
    }
    cntJ[J] += 1;
  }
  // species segments of the internal radial row
  int run = baseRs;
  for (int t = 0; t < T; ++t) {
    int c = cntJ[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) segR[a * (T + 1) + t] = run;
    run += c;
  }
  if (lane == 0) segR[a * (T + 1) + T] = run;
  run = baseAs;
  for (int t = 0; t < T; ++t) {
    int c = cntJA[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) segA[a * (T + 1) + t] = run;
    run += c;
  }
  if (lane == 0) segA[a * (T + 1) + T] = run;
}

// Final layout of the internal angular list: every (atom, J) segment is padded to a multiple of 4 pairs so that the
// 4-pair register tiles of the angular kernels never straddle a segment.  A dummy is float4(2 rcA, 0, 0, bits(a))
// : the basis functions clamp d / rc at 1, where f_k = f_k' = 0 exactly, so a dummy contributes exactly nothing.
// Only the two moment sweeps use the padded list; the force and gather kernels (lane = pair) keep the unpadded one.
// Warp per atom.
__global__ void k_pad_angular(int N, int T, const int *__restrict__ segAu, const int *__restrict__ segAp,
                              const float4 *__restrict__ pairAu, float4 *__restrict__ pairA, int *__restrict__ atomA,
                              float rdummy) {
  int a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (a >= N) return;
  for (int J = 0; J < T; ++J) {
    const int s0 = segAu[a * (T + 1) + J], n = segAu[a * (T + 1) + J + 1] - s0;
    const int d0 = segAp[a * (T + 1) + J], np = segAp[a * (T + 1) + J + 1] - d0;
    for (int e = lane; e < np; e += 32) {
      const bool real = e < n;
      pairA[d0 + e] = real ? pairAu[s0 + e] : make_float4(rdummy, 0.f, 0.f, __int_as_float(a));
      atomA[d0 + e] = a;
    }
  }
}

// reverse-pair index of the internal angular list: rev[p] = index of (j -> i, -shift).  Warp per atom.
__global__ void k_nbr_reverse(int N, const int *__restrict__ rowAs, const float4 *__restrict__ pairA,
                              const int *__restrict__ shA, int *__restrict__ revA) {
  int a = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (a >= N) return;
  for (int p = rowAs[a] + lane; p < rowAs[a + 1]; p += 32) {
    int b = __float_as_int(pairA[p].w);
    int sh = shA[p];
    int sa = ((sh >> 16) & 255) - 128, sb = ((sh >> 8) & 255) - 128, sc = (sh & 255) - 128;
    int want = ((128 - sa) << 16) | ((128 - sb) << 8) | (128 - sc);
    int found = -1;
    for (int o = rowAs[b]; o < rowAs[b + 1]; ++o)
      if (__float_as_int(pairA[o].w) == a && shA[o] == want) { found = o; break; }
    revA[p] = found;
  }
}
