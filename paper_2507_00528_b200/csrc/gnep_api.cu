// gnep_api.cu -- C ABI of libgnep_b200.so (include/gnep.h) and the host orchestration of the hot path:
// handle, resident batch, stream-ordered kernel sequence, CUDA graph of one epoch.
// No CPU fallback: every step of the path runs in the kernels of this directory.
#include "../../include/gnep.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "common.cuh"
#include "neighbor.cuh"
#include "cgrad_radial.cuh"   // includes net_tc_kernels.cuh (tensor-core network)
#include "pair_kernels.cuh"
#include "angular_kernels.cuh"
#include "angular_warp_kernels.cuh"
#include "reduce_kernels.cuh"
#include "peak_kernels.cuh"
#include "noalloc_kernels.cuh"
#include "net_small_kernels.cuh"
#include <mutex>

// Scratch of gnep_loss_terms_noalloc: per-structure partial sums + the ticket counter.  File-scope device memory
// (192 KiB + 256 B; every GPU that loads the library holds it until exit) so that the entry point allocates nothing.
// In host code this NAME is only a stand-in for the symbol: the kernel gets the device address that
// cudaGetSymbolAddress returns (noalloc_scratch(), once per device).
static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_SCRATCH_DOUBLES];

namespace {

thread_local std::string g_create_error;

// device address of g_noalloc_scratch on device `dev`: looked up once per device, with that device current
std::mutex g_noalloc_mu;
double *g_noalloc_ptr[64] = {};
cudaError_t noalloc_scratch(int dev, double **out) {
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e != cudaSuccess) return e;
    if (cur != dev && (e = cudaSetDevice(dev)) != cudaSuccess) return e;
    double *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, g_noalloc_scratch);
    if (cur != dev) cudaSetDevice(cur);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_noalloc_ptr[dev] = p;
  }
  *out = g_noalloc_ptr[dev];
  return cudaSuccess;
}

struct Phase { const char *name; cudaEvent_t ev; };

}  // namespace

struct gnep_handle {
  gnep_model_spec spec{};
  DevSpec ds{};
  cudaStream_t stream = nullptr;
  bool own_stream = false;
  bool shares_state = false;   // gnep_create_shared: theta, grad, m, v, q_scale, step belong to the parent
  mutable std::string err;
  int device = 0;
  int num_sms = 148;
  // parameters and optimiser
  float *theta = nullptr, *grad = nullptr, *m = nullptr, *v = nullptr, *qscale = nullptr;
  long long *step_dev = nullptr;
  float *terms = nullptr, *scales = nullptr;   // device: 5 loss terms, 4 seed multipliers
  float *lr_dev = nullptr;                     // device: learning rate read by k_adam
  float *h_terms = nullptr;                    // pinned host
  // batch
  bool loaded = false;
  int N = 0, S = 0;
  int64_t nR = 0, nA = 0;
  int hasE = 0, hasF = 0, hasV = 0;
  double Zloc[3] = {0, 0, 0};                // normalisers of the resident batch: sum w_e, sum w_f N_s, sum w_v (R40)
  double Zjob[3] = {-1, -1, -1};             // job-wide normalisers when structures are sharded over ranks (< 0: unset)
  double l2_share = 1.0;
  double *wgt = nullptr;                     // device [3][S]: per-structure weights of the three loss terms
  std::vector<int> host_aoff;                // atom offsets of the resident batch (for the weight normalisers)
  bool eval_local = false;                   // set while gnep_evaluate runs: RMSEs of the resident batch, whatever the job norm
  std::vector<void *> batch_allocs;
  int *perm = nullptr, *type_s = nullptr, *struct_s = nullptr, *segR = nullptr;
  // angular moment kernels, two mappings: warp tiles over a padded pair list (l_max <= 4, the fast
  // path) or slot-group tiles of 32 atoms (any l_max; always used above 4)
  bool tile_path = false;
  int *tilesA = nullptr;       // slot-group path: 32 atoms of one central species per tile, sorted by neighbour counts; -1 = idle lane
  int n_tilesA = 0, grid_adj = 0, grid_cg = 0, occ_adj = 1, occ_cg = 1, occ_S = 4;
  bool fuse_adam = false; float fuse_b1 = 0.f, fuse_b2 = 0.f, fuse_eps = 0.f;   // set while gnep_train_epochs captures its graph
  bool net_small = false;                  // small batches: the network on plain FMAs, warp per atom (net_small_kernels.cuh)
  int rad_lanes = RAD_SPLIT;               // lanes per atom of the split radial sweeps
  bool rad_split = false;                  // radial a3/a5 with RAD_SPLIT lanes per atom (small batches)
  int ta_ang = ANG_TA, ta_frc = FRC_TA;   // atoms per warp of the warp-tile sweeps: fewer for small batches, so that every SM gets warps
  int *segA = nullptr, *atomA = nullptr;   // warp-tile path: angular list with every (atom, J) segment padded to 4 pairs
  float4 *pairA = nullptr;
  int *rowAu = nullptr, *segAu = nullptr, *atomAu = nullptr, *revAu = nullptr;   // angular list
  float4 *pairAu = nullptr;
  float4 *pairR = nullptr;
  int64_t *exp_row[2] = {nullptr, nullptr};
  int *exp_j[2] = {nullptr, nullptr}, *exp_sh[2] = {nullptr, nullptr};
  int *srange = nullptr;
  double *Eref = nullptr, *Wref = nullptr;
  float *Fref_s = nullptr;
  SpeciesMap sm{};
  ReduceMap rm{};
  int n_cta_net = 0, n_chunks = 0, n_gw = 0;
  // per-atom state
  float *q = nullptr, *Sn = nullptr, *x = nullptr, *Ei = nullptr, *Ep = nullptr, *etil = nullptr, *M1 = nullptr,
        *M2 = nullptr, *D = nullptr, *Tn = nullptr, *A1 = nullptr, *A2 = nullptr, *Beta = nullptr, *gbar = nullptr, *pbuf = nullptr, *eat = nullptr, *Wat = nullptr;
  float4 *Fat = nullptr, *fpair = nullptr, *u = nullptr;
  double *Es = nullptr, *Ws = nullptr, *parts = nullptr;
  float *e_s = nullptr, *omega = nullptr;
  float *partialCR = nullptr, *partialCA = nullptr, *partialW = nullptr, *partialB = nullptr;
  // bookkeeping
  int64_t launches = 0;
  cudaGraphExec_t graph = nullptr;
  float g_lr = 0, g_b1 = 0, g_b2 = 0, g_eps = 0;
  int64_t graph_launches = 0;
  bool prof = false;
  std::vector<Phase> phases;
  std::vector<const char *> phase_names;
  std::vector<float> phase_ms;
};

namespace {

int fail(const gnep_handle *h, int code, const std::string &msg) {
  if (h) h->err = msg; else g_create_error = msg;
  return code;
}

#define CK(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess)                                                                         \
      return fail(h, e_ == cudaErrorMemoryAllocation ? GNEP_ENOMEM : GNEP_ECUDA,                   \
                  std::string(#call) + ": " + cudaGetErrorString(e_));                             \
  } while (0)

#define RET_IF(expr)            \
  do {                          \
    int rc_ = (expr);           \
    if (rc_ != GNEP_OK) return rc_; \
  } while (0)

int padded_basis(int K) {
  const int sizes[] = {4, 6, 8, 12, 16};
  for (int s : sizes) if (K <= s) return s;
  return -1;
}

#define DISPATCH_KT(KP, ...)                                    \
  switch (KP) {                                                 \
    case 4: { constexpr int KT = 4; __VA_ARGS__; } break;       \
    case 6: { constexpr int KT = 6; __VA_ARGS__; } break;       \
    case 8: { constexpr int KT = 8; __VA_ARGS__; } break;       \
    case 12: { constexpr int KT = 12; __VA_ARGS__; } break;     \
    default: { constexpr int KT = 16; __VA_ARGS__; } break;     \
  }

// angular kernels: basis size padded to 4, 8 or 16 (32 / KT functions per lane-sum chunk), harmonics compiled for
// l_max <= 4 (24 slots, 4 slot groups) and l_max <= 8 (80 slots, 14 slot groups)
int padded_basis_ang(int K) { return K <= 4 ? 4 : K <= 8 ? 8 : 16; }
#define DISPATCH_KA(KP, ...)                                    \
  switch (KP) {                                                 \
    case 4: { constexpr int KT = 4; __VA_ARGS__; } break;       \
    case 8: { constexpr int KT = 8; __VA_ARGS__; } break;       \
    default: { constexpr int KT = 16; __VA_ARGS__; } break;     \
  }
// warp-tile kernels: n (angular radial functions) padded to the register-array size of the sweeps
#define DISPATCH_NQ(NA_, ...)                                   \
  if ((NA_) <= 10) { constexpr int NQ = 10; __VA_ARGS__; }      \
  else { constexpr int NQ = 16; __VA_ARGS__; }
#define DISPATCH_SPLIT(L_, ...)                                          \
  if ((L_) == RAD_SPLIT_WIDE) { constexpr int SPLIT = RAD_SPLIT_WIDE; __VA_ARGS__; } \
  else { constexpr int SPLIT = RAD_SPLIT; __VA_ARGS__; }
#define DISPATCH_B5(U5_, ...)                                   \
  if (U5_) { constexpr bool B5 = true; __VA_ARGS__; }           \
  else { constexpr bool B5 = false; __VA_ARGS__; }
#define DISPATCH_TMAX(T_, ...)                                  \
  if ((T_) <= 2) { constexpr int TMAX = 2; __VA_ARGS__; }       \
  else { constexpr int TMAX = 4; __VA_ARGS__; }
#define DISPATCH_ANG(d_, ...)                                               \
  if ((d_).L <= 4) { constexpr int LMAX = 4; DISPATCH_KA((d_).KAp, __VA_ARGS__) } \
  else { constexpr int LMAX = 8; DISPATCH_KA((d_).KAp, __VA_ARGS__) }

template <class T>
int dalloc(gnep_handle *h, T **p, size_t n, bool batch) {
  void *q = nullptr;
  CK(cudaMalloc(&q, std::max<size_t>(n, 1) * sizeof(T)));
  *p = (T *)q;
  if (batch) h->batch_allocs.push_back(q);
  return GNEP_OK;
}

void free_batch(gnep_handle *h) {
  for (void *p : h->batch_allocs) cudaFree(p);
  h->batch_allocs.clear();
  h->loaded = false;
  if (h->graph) { cudaGraphExecDestroy(h->graph); h->graph = nullptr; }
}

// ---- dynamic shared memory sizes (bytes) --------------------------------------------------------
size_t smem_radial(const DevSpec &d) { return sizeof(float) * (d.T * d.T * d.NR * d.KRp); }
int ang_lmax(const DevSpec &d) { return d.L <= 4 ? 4 : 8; }               // harmonics instantiation of the slot-group kernels
int ang_warps(const DevSpec &d) { return ang_groups(ang_lmax(d)); }       // warps per CTA (the model uses ang_groups(L) slot groups)
size_t smem_ang_fwd(const DevSpec &d) { return sizeof(float) * ang_fwd_smem_floats(d.T, d.NA, d.KAp, ang_lmax(d), d.Ndes - d.NR); }
size_t smem_ang_force(const DevSpec &d) { return sizeof(float) * (((d.T * d.T * d.NA * d.KAp + 3) & ~3) + FRC_WARPS * FRC_TA * d.NA * d.nlmS); }
size_t smem_ang_adj(const DevSpec &d) { return sizeof(float) * ang_adj_smem_floats(d.T, d.NA, d.KAp, ang_lmax(d), d.Ndes - d.NR); }
size_t smem_cgrad_ang(const DevSpec &d) { return sizeof(float) * ang_cgrad_smem_floats(d.T, d.NA, d.KAp, ang_lmax(d), d.Ndes - d.NR); }
size_t smem_angw_fwd(const DevSpec &d) {
  return sizeof(float) * (d.T * d.T * d.KAp * ANG_NQ + ANG_WARPS * ((d.KAp + ANGW_NLM) * ANG_LD + d.T * d.KAp * ANGW_NLM + ANG_NQ * ANGW_NLM + ANG_SEGS));
}
size_t smem_angw_S(const DevSpec &d) { return sizeof(float) * (size_t)angw_S_smem_floats(d.T, d.NA, d.KAp, d.NR, d.KRp); }
size_t smem_angw_adj(const DevSpec &d) {
  return sizeof(float) * (d.T * d.T * d.KAp * ANG_NQ + ANG_WARPS * ((2 * d.KAp + 2 * ANGW_NLM) * ANG_LD + d.T * d.KAp * ANGW_NLM + ANG_NQ * ANGW_NLM + ANG_SEGS));
}
size_t smem_angw_cgrad(const DevSpec &d) {
  return sizeof(float) * ANG_WARPS * (((d.T * d.T * d.NA * d.KAp + 3) & ~3) + 2 * ((d.NA * ANGW_NLM + 3) & ~3));
}
size_t smem_net_fwd(const DevSpec &d) { return net_tc_smem_bytes(d, false); }
size_t smem_net_bwd(const DevSpec &d) { return net_tc_smem_bytes(d, true); }
size_t smem_gradw(const DevSpec &d) { return gradw_smem_bytes(d); }
size_t smem_cgrad_rad(const DevSpec &d) { return cgrad_radial_smem_bytes(d); }

template <class K>
int set_smem(gnep_handle *h, K kernel, size_t bytes) {
  if (bytes > 227 * 1024) return fail(h, GNEP_EINVAL, "model too large for shared memory staging (n_neurons x n_descriptors)");
  // the attribute is process-wide per kernel: always the hardware maximum, so that a later, smaller model never lowers
  // the limit under a live handle (each launch still asks only for what its own model needs)
  CK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
  return GNEP_OK;
}

int configure_kernels(gnep_handle *h) {
  const DevSpec &d = h->ds;
  DISPATCH_KT(d.KRp, RET_IF(set_smem(h, k_radial_fwd<KT>, smem_radial(d))); RET_IF(set_smem(h, k_radial_adj<KT>, smem_radial(d))); { auto k8 = k_radial_adj_split<KT, RAD_SPLIT>; auto k32 = k_radial_adj_split<KT, RAD_SPLIT_WIDE>; RET_IF(set_smem(h, k8, smem_radial(d))); RET_IF(set_smem(h, k32, smem_radial(d))); }
              RET_IF(set_smem(h, k_radial_q<KT>, smem_radial(d))));
  DISPATCH_ANG(d, auto kf = k_angular_fwd<KT, LMAX>; auto ka = k_angular_adj<KT, LMAX>; auto kc = k_cgrad_angular<KT, LMAX>;
               auto kp = k_angular_force<KT, LMAX>;
               RET_IF(set_smem(h, kf, smem_ang_fwd(d))); RET_IF(set_smem(h, ka, smem_ang_adj(d)));
               RET_IF(set_smem(h, kc, smem_cgrad_ang(d))); RET_IF(set_smem(h, kp, smem_ang_force(d)));
               // persistent grids of the two accumulating kernels: one resident wave
               int occ = 0;
               CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, ka, 32 * ang_warps(d), smem_ang_adj(d)));
               h->occ_adj = std::max(occ, 1);
               CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kc, 32 * ang_warps(d), smem_cgrad_ang(d)));
               h->occ_cg = std::max(occ, 1));
  if (!h->tile_path) {
    DISPATCH_KA(d.KAp, DISPATCH_B5(d.use5, auto kc5 = k_angw_cgrad<KT, B5>; RET_IF(set_smem(h, kc5, smem_angw_cgrad(d)))); DISPATCH_TMAX(d.T, auto ks = k_angw_S<KT, TMAX>; RET_IF(set_smem(h, ks, smem_angw_S(d)));
                              int occ = 0;
                              CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, ks, ANG_WARPS * 32, smem_angw_S(d)));
                              h->occ_S = std::max(occ, 1));
                DISPATCH_NQ(d.NA, auto kf = k_angw_fwd<KT, NQ>; RET_IF(set_smem(h, kf, smem_angw_fwd(d)));
                            DISPATCH_B5(d.use5, auto ka = k_angw_adj<KT, NQ, B5>; RET_IF(set_smem(h, ka, smem_angw_adj(d))))));
  }
  {   // TMEM budget of one k_net_tc warpgroup (256 columns): D1 + max(D1 corrections, D2 + D2 corrections)
    const NetDims nd = net_dims(d);
    if (nd.NnP + std::max(nd.NnP, 2 * nd.NdN) > 256) return fail(h, GNEP_EINVAL, "model too large for tensor memory (n_neurons, n_descriptors)");
  }
  RET_IF(set_smem(h, k_net_tc<false>, smem_net_fwd(d)));
  RET_IF(set_smem(h, k_net_tc<true>, smem_net_bwd(d)));
  if (gradw_nraw(d) < 2) return fail(h, GNEP_EINVAL, "model too large for shared memory staging (n_descriptors)");
  RET_IF(set_smem(h, k_gradw_tc, smem_gradw(d)));
  RET_IF(set_smem(h, k_cgrad_radial, smem_cgrad_rad(d)));
  RET_IF(set_smem(h, k_net_small_fwd, 0)); RET_IF(set_smem(h, k_net_small_bwd, 0));   // (used only when the model fits: net_small)
  return GNEP_OK;
}

void mark(gnep_handle *h, const char *name) {
  if (!h->prof) return;
  Phase p; p.name = name;
  cudaEventCreate(&p.ev);
  cudaEventRecord(p.ev, h->stream);
  h->phases.push_back(p);
}
void prof_begin(gnep_handle *h) {
  if (!h->prof) return;
  for (auto &p : h->phases) cudaEventDestroy(p.ev);
  h->phases.clear();
  mark(h, "begin");
}
void prof_collect(gnep_handle *h) {
  if (!h->prof || h->phases.empty()) return;
  cudaEventSynchronize(h->phases.back().ev);
  h->phase_names.clear(); h->phase_ms.clear();
  for (size_t i = 1; i < h->phases.size(); ++i) {
    float ms = 0.f;
    cudaEventElapsedTime(&ms, h->phases[i - 1].ev, h->phases[i].ev);
    h->phase_names.push_back(h->phases[i].name);
    h->phase_ms.push_back(ms);
  }
}

inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

#define LAUNCH(h, kern, grid, block, smem, ...)                       \
  do {                                                                \
    if ((grid) > 0) {                                                 \
      kern<<<(grid), (block), (smem), (h)->stream>>>(__VA_ARGS__);   \
      (h)->launches++;                                                \
    }                                                                 \
  } while (0)

// ---- the forward half: descriptors, network, forces, per-structure sums (rows a1-a4) --------------
// Geometry-only moments of the resident batch: M1[J][k] = sum_j f_k(d_ij) and, on the warp-tile path,
// A1[J][k][lm] = sum_j f_k B_lm.  They do not depend on theta and positions are fixed during training, so the pair
// sweeps that build them run ONCE, at the end of gnep_load_batch; the epoch's descriptor pass contracts them with c.
int enqueue_geometry_moments(gnep_handle *h) {
  const DevSpec &d = h->ds;
  DISPATCH_KT(d.KRp, LAUNCH(h, k_radial_fwd<KT>, cdiv(h->N, RAD_THREADS), RAD_THREADS, smem_radial(d), d, h->N, h->type_s, h->segR, h->pairR, h->theta, h->q, h->M1));
  if (!h->tile_path) {
    DISPATCH_KA(d.KAp, DISPATCH_NQ(d.NA, auto kf = k_angw_fwd<KT, NQ>; LAUNCH(h, kf, cdiv(h->N, ANG_WARPS * h->ta_ang), ANG_WARPS * 32, smem_angw_fwd(d), d, h->N, h->ta_ang, h->type_s, h->segA, h->pairA, h->theta, h->q, h->Sn, h->A1)));
  }
  return GNEP_OK;
}

int enqueue_descriptors(gnep_handle *h) {
  const DevSpec &d = h->ds;
  if (!h->tile_path) {   // one kernel: radial and angular contractions with the resident moments
    DISPATCH_KA(d.KAp, DISPATCH_TMAX(d.T, auto ks = k_angw_S<KT, TMAX>; LAUNCH(h, ks, std::max(1, std::min(cdiv(h->N, 2 * ANG_WARPS), h->occ_S * h->num_sms)), ANG_WARPS * 32, smem_angw_S(d), d, h->N, h->type_s, h->theta, h->M1, h->A1, h->q, h->Sn)));
    mark(h, "a1_descriptor_contraction");
    return GNEP_OK;
  }
  DISPATCH_KT(d.KRp, LAUNCH(h, k_radial_q<KT>, cdiv(h->N, RAD_THREADS), RAD_THREADS, smem_radial(d), d, h->N, h->type_s, h->theta, h->M1, h->q));
  mark(h, "a1_radial_descriptor");
  DISPATCH_ANG(d, auto kf = k_angular_fwd<KT, LMAX>; LAUNCH(h, kf, h->n_tilesA, 32 * ang_warps(d), smem_ang_fwd(d), d, h->n_tilesA, h->tilesA, h->type_s, h->segAu, h->pairAu, h->theta, h->q, h->Sn, h->A1));
  mark(h, "a1_angular_descriptor");
  return GNEP_OK;
}

LossCfg loss_cfg(const gnep_handle *h) {
  LossCfg lc;
  lc.S = h->S; lc.N = h->N; lc.T = h->ds.T; lc.P = h->ds.P;
  lc.hasE = h->hasE; lc.hasF = h->hasF; lc.hasV = h->hasV; lc.loss_mode = h->ds.loss_mode;
  lc.lam_e = h->spec.lambda_e; lc.lam_f = h->spec.lambda_f; lc.lam_v = h->spec.lambda_v; lc.lam_2 = h->spec.lambda_2;
  const bool job = h->Zjob[0] >= 0 && !h->eval_local;   // gnep_evaluate always normalises by the resident batch itself
  const double *Z = job ? h->Zjob : h->Zloc;
  lc.ZE = Z[0]; lc.ZF = Z[1]; lc.ZV = Z[2]; lc.l2_share = job ? h->l2_share : 1.0;
  lc.rZE = Z[0] > 0 ? 1.0 / Z[0] : 0.0; lc.rZF3 = Z[1] > 0 ? 1.0 / (3.0 * Z[1]) : 0.0; lc.rZV6 = Z[2] > 0 ? 1.0 / (6.0 * Z[2]) : 0.0;
  lc.rP = lc.P > 0 ? 1.0 / (double)lc.P : 0.0;
  return lc;
}

int enqueue_forward(gnep_handle *h) {
  const DevSpec &d = h->ds;
  const bool fuse_desc = h->net_small && !h->tile_path;   // small batches: the descriptor contraction inside the network kernel
  if (!fuse_desc) RET_IF(enqueue_descriptors(h));
  if (h->net_small) {
    LAUNCH(h, k_net_small_fwd, h->n_gw, NS_THREADS, sizeof(float) * net_small_fwd_floats(d), d, h->sm, h->theta, h->qscale, h->q, h->x, h->Ei, h->Ep, h->etil,
           fuse_desc ? h->A1 : (const float *)nullptr, h->M1, h->Sn);
    if (fuse_desc) mark(h, "a1_descriptor_contraction");
  } else {
    LAUNCH(h, k_net_tc<false>, h->n_cta_net, 256, smem_net_fwd(d), d, h->sm, h->theta, h->qscale, h->q, h->x, h->Ei, h->Ep, h->etil,
           (const int *)nullptr, (const float *)nullptr, (const float *)nullptr, (float *)nullptr, (float *)nullptr);
  }
  mark(h, "a2_network_forward");
  DISPATCH_ANG(d, auto kp = k_angular_force<KT, LMAX>; LAUNCH(h, kp, cdiv(h->N, FRC_WARPS * h->ta_frc), FRC_WARPS * 32, smem_ang_force(d), d, h->N, h->ta_frc, h->type_s, h->segAu, h->atomAu, h->pairAu, h->theta, h->Ep, h->Sn, h->tile_path ? h->Beta : (float *)nullptr, h->fpair));
  mark(h, "a3_angular_force");
  // radial forces + the gather of the angular pair forces (thread per atom): writes F_i, W_i once
  if (h->rad_split) {
    DISPATCH_KT(d.KRp, DISPATCH_SPLIT(h->rad_lanes, auto kf = k_radial_force_split<KT, SPLIT>; LAUNCH(h, kf, cdiv((int64_t)h->N * SPLIT, RAD_THREADS), RAD_THREADS, 0, d, h->N, h->type_s, h->segR, h->pairR, h->etil,
                              h->segAu, h->revAu, h->pairAu, h->fpair, h->Fat, h->Wat)));
  } else {
    DISPATCH_KT(d.KRp, LAUNCH(h, k_radial_force<KT>, cdiv(h->N, RAD_THREADS), RAD_THREADS, 0, d, h->N, h->type_s, h->segR, h->pairR, h->etil,
                              h->segAu, h->revAu, h->pairAu, h->fpair, h->Fat, h->Wat));
  }
  mark(h, "a3_radial_force");
  // terms[5..6] = the Adam bias corrections of this step, terms[7] = the ticket counter of k_struct_reduce (zero at rest)
  const AdamPre ap = {h->step_dev, h->terms + 5, h->fuse_b1, h->fuse_b2, std::log((double)h->fuse_b1), std::log((double)h->fuse_b2), h->fuse_adam ? 1 : 0};
  if (h->S > 0) {
    LAUNCH(h, k_struct_reduce, h->S <= 4 ? 1 : h->S + LOSS_T2_CTAS, 128, 0, loss_cfg(h), h->srange, h->Ei, h->Fat, h->Wat, h->Eref, h->Fref_s, h->Wref, h->wgt, h->Es, h->Ws, h->e_s, h->u, h->omega, h->parts,
           (unsigned *)(h->terms + 7), h->theta, h->terms, h->scales, ap);
  } else {
    LAUNCH(h, k_loss_final, 1, 128, 0, loss_cfg(h), h->parts, h->theta, h->terms, h->scales, ap);
  }
  mark(h, "a4_loss_and_seeds");
  return GNEP_OK;
}

// ---- the backward half (rows a5-a8) ----------------------------------------------------------------
int enqueue_backward(gnep_handle *h) {
  const DevSpec &d = h->ds;
  if (h->rad_split) {
    DISPATCH_KT(d.KRp, DISPATCH_SPLIT(h->rad_lanes, auto ka = k_radial_adj_split<KT, SPLIT>; LAUNCH(h, ka, cdiv((int64_t)h->N * SPLIT, RAD_THREADS), RAD_THREADS, smem_radial(d), d, h->N, h->type_s, h->struct_s, h->segR, h->pairR, h->theta, h->u, h->omega, h->scales, h->D, h->M2)));
  } else {
    DISPATCH_KT(d.KRp, LAUNCH(h, k_radial_adj<KT>, cdiv(h->N, RAD_THREADS), RAD_THREADS, smem_radial(d), d, h->N, h->type_s, h->struct_s, h->segR, h->pairR, h->theta, h->u, h->omega, h->scales, h->D, h->M2));
  }
  mark(h, "a5_radial_adjoint");
  if (!h->tile_path) {
    DISPATCH_KA(d.KAp, DISPATCH_NQ(d.NA, DISPATCH_B5(d.use5, auto ka = k_angw_adj<KT, NQ, B5>; LAUNCH(h, ka, cdiv(h->N, ANG_WARPS * h->ta_ang), ANG_WARPS * 32, smem_angw_adj(d), d, h->N, h->ta_ang, h->type_s, h->struct_s, h->segA, h->atomA, h->pairA, h->theta, h->u, h->omega, h->scales, h->Sn, h->Tn, h->A2, h->D))));
  } else
  DISPATCH_ANG(d, auto ka = k_angular_adj<KT, LMAX>; LAUNCH(h, ka, h->grid_adj, 32 * ang_warps(d), smem_ang_adj(d), d, h->n_tilesA, h->tilesA, h->type_s, h->struct_s, h->segAu, h->pairAu, h->theta, h->u, h->omega, h->scales, h->Sn, h->Beta, h->Tn, h->D, h->partialCA));
  mark(h, "a5_angular_adjoint");
  if (h->net_small) {   // network backward and its parameter-gradient partials in one launch
    LAUNCH(h, k_net_small_bwd, h->n_gw, NS_THREADS, sizeof(float) * net_small_bwd_floats(d), d, h->sm, h->theta, h->qscale, h->q, h->D, h->x, h->Ep,
           h->struct_s, h->e_s, h->scales, h->M1, h->M2, h->gbar, h->partialW, h->partialB, h->partialCR);
    mark(h, "a6_network_backward");
  } else {
    LAUNCH(h, k_net_tc<true>, h->n_cta_net, 256, smem_net_bwd(d), d, h->sm, h->theta, h->qscale, h->D, h->x, h->eat, h->Ep, (float *)nullptr,
           h->struct_s, h->e_s, h->scales, h->pbuf, h->gbar);
    mark(h, "a6_network_backward");
    LAUNCH(h, k_gradw_tc, h->n_gw, GW_THREADS, smem_gradw(d), d, h->sm, gradw_nraw(d), h->theta, h->qscale, h->eat, h->q, h->D, h->x, h->pbuf, h->partialW, h->partialB);
  }
  mark(h, "a6_w0_gradient");
  if (!h->net_small)   // (the small-batch network backward forms these partials itself)
    LAUNCH(h, k_cgrad_radial, h->n_chunks, CR_THREADS, smem_cgrad_rad(d), d, h->sm, h->gbar, h->Ep, h->M1, h->M2, h->partialCR);
  mark(h, "a7_radial_cgrad");
  if (!h->tile_path) {
    DISPATCH_KA(d.KAp, DISPATCH_B5(d.use5, auto kc5 = k_angw_cgrad<KT, B5>; LAUNCH(h, kc5, h->grid_cg, ANG_WARPS * 32, smem_angw_cgrad(d), d, h->N, h->type_s, h->Ep, h->gbar, h->Sn, h->Tn, h->A1, h->A2, h->partialCA)));
  } else
  DISPATCH_ANG(d, auto kc = k_cgrad_angular<KT, LMAX>; LAUNCH(h, kc, h->grid_cg, 32 * ang_warps(d), smem_cgrad_ang(d), d, h->n_tilesA, h->tilesA, h->type_s, h->segAu, h->Ep, h->gbar, h->Sn, h->Tn, h->A1,
                                                          h->partialCA + (size_t)h->grid_adj * ang_warps(d) * d.T * d.T * d.NA * d.KAp));
  mark(h, "a7_angular_cgrad");
  // inside a captured training step the Adam update (a9) rides on the reduction: the thread that sums a parameter's partials updates it
  const AdamFuse af = {h->m, h->v, h->terms + 5, h->lr_dev, h->fuse_b1, h->fuse_b2, h->fuse_eps, h->fuse_adam ? 1 : 0};
  LAUNCH(h, k_grad_reduce, cdiv(d.P, 8), 256, 0, d, h->rm, (float)h->l2_share, h->theta, h->scales, h->partialCR, h->partialCA, h->partialW, h->partialB, h->grad, af);
  mark(h, "a8_grad_reduce");
  return GNEP_OK;
}

void set_lr(gnep_handle *h, float lr) { LAUNCH(h, k_set_scalar, 1, 1, 0, h->lr_dev, lr); }
int enqueue_adam(gnep_handle *h, float b1, float b2, float eps) {
  LAUNCH(h, k_adam, cdiv(h->ds.P, 256), 256, 0, h->ds.P, h->theta, h->m, h->v, h->grad, h->step_dev, h->lr_dev, b1, b2, eps);
  LAUNCH(h, k_step_inc, 1, 1, 0, h->step_dev);
  mark(h, "a9_adam");
  return GNEP_OK;
}

int check_launch(gnep_handle *h) {
  CK(cudaGetLastError());
  return GNEP_OK;
}

// copy helper: caller buffer <-> device
int copy_in(gnep_handle *h, void *dst, const void *src, size_t bytes, int is_device) {
  CK(cudaMemcpyAsync(dst, src, bytes, is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
  if (!is_device) CK(cudaStreamSynchronize(h->stream));   // pageable host memory may be reused by the caller
  return GNEP_OK;
}
int copy_out(const gnep_handle *hc, void *dst, const void *src, size_t bytes, int is_device) {
  gnep_handle *h = const_cast<gnep_handle *>(hc);
  CK(cudaMemcpyAsync(dst, src, bytes, is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  return GNEP_OK;
}

int fetch_terms(gnep_handle *h, float *loss_terms) {
  CK(cudaMemcpyAsync(h->h_terms, h->terms, 5 * sizeof(float), cudaMemcpyDeviceToHost, h->stream));
  CK(cudaStreamSynchronize(h->stream));
  prof_collect(h);
  for (int i = 0; i < 5; ++i) loss_terms[i] = h->h_terms[i];
  if (!std::isfinite(loss_terms[0])) return fail(h, GNEP_ENONFINITE, "loss is not finite");
  return GNEP_OK;
}

struct HostGeo { double h[3]; };

int cell_geometry(const double *c, double *inv, double *hh) {
  const double *a = c, *b = c + 3, *cc = c + 6;
  auto cross = [](const double *u, const double *v, double *o) {
    o[0] = u[1] * v[2] - u[2] * v[1]; o[1] = u[2] * v[0] - u[0] * v[2]; o[2] = u[0] * v[1] - u[1] * v[0];
  };
  auto dot = [](const double *u, const double *v) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; };
  double bxc[3], cxa[3], axb[3];
  cross(b, cc, bxc); cross(cc, a, cxa); cross(a, b, axb);
  double V = dot(a, bxc);
  if (!(std::fabs(V) > 0.0) || !std::isfinite(V)) return -1;
  hh[0] = std::fabs(V) / std::sqrt(dot(bxc, bxc));
  hh[1] = std::fabs(V) / std::sqrt(dot(cxa, cxa));
  hh[2] = std::fabs(V) / std::sqrt(dot(axb, axb));
  for (int k = 0; k < 3; ++k) { inv[k] = bxc[k] / V; inv[3 + k] = cxa[k] / V; inv[6 + k] = axb[k] / V; }
  return 0;
}

}  // namespace

// ====================================================================================================
extern "C" {

const char *gnep_last_error(const gnep_handle *h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int gnep_create(const gnep_model_spec *spec, void *cuda_stream, gnep_handle **out) {
  gnep_handle *h = nullptr;   // errors before the handle exists go to the thread-local string
  if (!spec || !out) return fail(h, GNEP_EINVAL, "null spec or out");
  *out = nullptr;
  const gnep_model_spec &s = *spec;
  if (s.n_species < 1 || s.n_species > GNEP_MAX_SPECIES) return fail(h, GNEP_EINVAL, "n_species out of range");
  if (s.n_radial < 1 || s.n_radial > GNEP_MAX_NFUNC || s.n_angular < 1 || s.n_angular > GNEP_MAX_NFUNC)
    return fail(h, GNEP_EINVAL, "n_radial / n_angular out of range");
  if (s.n_basis_radial < 1 || s.n_basis_radial > GNEP_MAX_BASIS || s.n_basis_angular < 1 || s.n_basis_angular > GNEP_MAX_BASIS)
    return fail(h, GNEP_EINVAL, "basis size out of range");
  if (!(s.rc_radial > 0) || !(s.rc_angular > 0) || s.rc_angular > s.rc_radial) return fail(h, GNEP_EINVAL, "need 0 < rc_angular <= rc_radial");
  if (s.l_max < 1 || s.l_max > GNEP_LMAX) return fail(h, GNEP_EINVAL, "l_max must be 1..8");
  if (s.use_4body && s.l_max < 2) return fail(h, GNEP_EINVAL, "use_4body needs l_max >= 2");
  if (s.n_neurons < 1 || s.n_neurons > GNEP_MAX_NEURONS) return fail(h, GNEP_EINVAL, "n_neurons out of range");
  if (s.loss_mode != 0 && s.loss_mode != 1) return fail(h, GNEP_EINVAL, "loss_mode must be 0 or 1");
  if (s.lambda_e < 0 || s.lambda_f < 0 || s.lambda_v < 0 || s.lambda_2 < 0) return fail(h, GNEP_EINVAL, "negative loss weight");
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    cudaGetLastError();
    return fail(h, GNEP_ECUDA, "no CUDA device (this library has no CPU fallback)");
  }
  if (prop.major != 10) return fail(h, GNEP_ECUDA, "device is not compute capability 10.x (built for sm_100a only)");
  h = new (std::nothrow) gnep_handle();
  if (!h) return fail(nullptr, GNEP_ENOMEM, "out of host memory");
  h->spec = s; h->spec.q_scale = nullptr;
  h->device = dev; h->num_sms = prop.multiProcessorCount;
  DevSpec &d = h->ds;
  d.T = s.n_species; d.NR = s.n_radial; d.KR = s.n_basis_radial; d.NA = s.n_angular; d.KA = s.n_basis_angular;
  d.L = s.l_max; d.use4 = s.use_4body ? 1 : 0; d.use5 = s.use_5body ? 1 : 0; d.Nn = s.n_neurons; d.NnS = (d.Nn + 15) & ~15;
  d.Ndes = d.NR + d.NA * d.L + (d.use4 ? d.NA : 0) + (d.use5 ? d.NA : 0);
  d.nlmS = d.L <= 4 ? 24 : 88;   // 24 / 80 slots; rows are whole 32-byte pieces
  d.KRp = padded_basis(d.KR); d.KAp = padded_basis_ang(d.KA);
  d.offA = d.T * d.T * d.NR * d.KR;
  d.offNet = d.offA + d.T * d.T * d.NA * d.KA;
  d.netSize = d.Nn * d.Ndes + 2 * d.Nn + 1;
  d.P = d.offNet + d.T * d.netSize;
  d.ldW = d.Ndes | 1;
  d.loss_mode = s.loss_mode;
  d.rcRinv = (float)(1.0 / s.rc_radial); d.rcAinv = (float)(1.0 / s.rc_angular);
  d.lam_e = (float)s.lambda_e; d.lam_f = (float)s.lambda_f; d.lam_v = (float)s.lambda_v; d.lam_2 = (float)s.lambda_2;
  auto bail = [&](int rc) { std::string e = h->err; gnep_destroy(h); g_create_error = e; return rc; };
  if (cuda_stream) h->stream = (cudaStream_t)cuda_stream;
  else {
    if (cudaStreamCreate(&h->stream) != cudaSuccess) { h->err = "cudaStreamCreate failed"; return bail(GNEP_ECUDA); }
    h->own_stream = true;
  }
  {   // GNEP_ANGULAR_MAPPING=groups forces the slot-group kernels for l_max <= 4 as well (they are the only ones above 4)
    const char *m = getenv("GNEP_ANGULAR_MAPPING");
    h->tile_path = d.L > 4 || (m && std::string(m) == "groups");
  }
  int rc;
  if ((rc = configure_kernels(h)) != GNEP_OK) return bail(rc);
  if ((rc = dalloc(h, &h->theta, d.P, false)) || (rc = dalloc(h, &h->grad, d.P, false)) || (rc = dalloc(h, &h->m, d.P, false)) ||
      (rc = dalloc(h, &h->v, d.P, false)) || (rc = dalloc(h, &h->qscale, d.Ndes, false)) || (rc = dalloc(h, &h->step_dev, 1, false)) ||
      (rc = dalloc(h, &h->terms, 8, false)) || (rc = dalloc(h, &h->scales, 4, false)) || (rc = dalloc(h, &h->lr_dev, 1, false)))
    return bail(rc);
  if (cudaMallocHost((void **)&h->h_terms, 8 * sizeof(float)) != cudaSuccess) { h->err = "cudaMallocHost failed"; return bail(GNEP_ENOMEM); }
  std::vector<float> qs(d.Ndes, 1.f);
  if (s.q_scale) for (int i = 0; i < d.Ndes; ++i) qs[i] = s.q_scale[i];
  float ones[4] = {1.f, 1.f, 1.f, 1.f};
  if (cudaMemsetAsync(h->theta, 0, d.P * sizeof(float), h->stream) != cudaSuccess ||
      cudaMemsetAsync(h->grad, 0, d.P * sizeof(float), h->stream) != cudaSuccess ||
      cudaMemsetAsync(h->m, 0, d.P * sizeof(float), h->stream) != cudaSuccess ||
      cudaMemsetAsync(h->v, 0, d.P * sizeof(float), h->stream) != cudaSuccess ||
      cudaMemsetAsync(h->step_dev, 0, sizeof(long long), h->stream) != cudaSuccess ||
      cudaMemsetAsync(h->terms, 0, 8 * sizeof(float), h->stream) != cudaSuccess ||
      cudaMemcpyAsync(h->scales, ones, sizeof(ones), cudaMemcpyHostToDevice, h->stream) != cudaSuccess ||
      cudaMemcpyAsync(h->qscale, qs.data(), d.Ndes * sizeof(float), cudaMemcpyHostToDevice, h->stream) != cudaSuccess ||
      cudaStreamSynchronize(h->stream) != cudaSuccess) { h->err = "initialisation copies failed"; return bail(GNEP_ECUDA); }
  *out = h;
  return GNEP_OK;
}

int gnep_destroy(gnep_handle *h) {
  if (!h) return GNEP_OK;
  if (h->stream) cudaStreamSynchronize(h->stream);
  free_batch(h);
  for (auto &p : h->phases) cudaEventDestroy(p.ev);
  if (!h->shares_state) { cudaFree(h->theta); cudaFree(h->grad); cudaFree(h->m); cudaFree(h->v); cudaFree(h->qscale); cudaFree(h->step_dev); }
  cudaFree(h->terms); cudaFree(h->scales); cudaFree(h->lr_dev);
  if (h->h_terms) cudaFreeHost(h->h_terms);
  if (h->own_stream && h->stream) cudaStreamDestroy(h->stream);
  delete h;
  return GNEP_OK;
}

int gnep_create_shared(const gnep_handle *parent, gnep_handle **out) {
  if (!parent || !out) return fail(parent, GNEP_EINVAL, "null parent or out");
  gnep_model_spec s = parent->spec;
  s.q_scale = nullptr;
  gnep_handle *h = nullptr;
  int rc = gnep_create(&s, (void *)parent->stream, &h);
  if (rc != GNEP_OK) { parent->err = g_create_error; return rc; }
  cudaFree(h->theta); cudaFree(h->grad); cudaFree(h->m); cudaFree(h->v); cudaFree(h->qscale); cudaFree(h->step_dev);
  h->theta = parent->theta; h->grad = parent->grad; h->m = parent->m; h->v = parent->v; h->qscale = parent->qscale;
  h->step_dev = parent->step_dev;
  h->shares_state = true;
  *out = h;
  return GNEP_OK;
}

int gnep_lr_schedule(int64_t step, int64_t n_warmup, int64_t n_total, double lr_start, double lr_stop, double *lr) {
  if (!lr || n_total < 1 || n_warmup < 0 || n_warmup > n_total) return GNEP_EINVAL;
  const int64_t s = step < 0 ? 0 : (step > n_total ? n_total : step);
  if (s < n_warmup) *lr = lr_stop + (double)s / (double)n_warmup * (lr_start - lr_stop);
  else if (n_total == n_warmup) *lr = lr_start;
  else *lr = lr_stop + (lr_start - lr_stop) * 0.5 * (1.0 + std::cos(3.14159265358979323846 * (double)(s - n_warmup) / (double)(n_total - n_warmup)));
  return GNEP_OK;
}

int gnep_num_params(const gnep_handle *h, int64_t *P) {
  if (!h || !P) return fail(h, GNEP_EINVAL, "null argument");
  *P = h->ds.P;
  return GNEP_OK;
}
int gnep_num_descriptors(const gnep_handle *h, int32_t *n) {
  if (!h || !n) return fail(h, GNEP_EINVAL, "null argument");
  *n = h->ds.Ndes;
  return GNEP_OK;
}

int gnep_set_params(gnep_handle *h, const float *theta, int is_device) {
  if (!h || !theta) return fail(h, GNEP_EINVAL, "null argument");
  return copy_in(h, h->theta, theta, h->ds.P * sizeof(float), is_device);
}
int gnep_get_params(const gnep_handle *h, float *theta, int is_device) {
  if (!h || !theta) return fail(h, GNEP_EINVAL, "null argument");
  return copy_out(h, theta, h->theta, h->ds.P * sizeof(float), is_device);
}
int gnep_set_q_scale(gnep_handle *h, const float *q_scale) {
  if (!h || !q_scale) return fail(h, GNEP_EINVAL, "null argument");
  for (int i = 0; i < h->ds.Ndes; ++i)
    if (!std::isfinite(q_scale[i])) return fail(h, GNEP_EINVAL, "q_scale not finite");
  return copy_in(h, h->qscale, q_scale, h->ds.Ndes * sizeof(float), 0);
}

int gnep_get_opt_state(const gnep_handle *h, float *m, float *v, int64_t *step, int is_device) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (m) RET_IF(copy_out(h, m, h->m, h->ds.P * sizeof(float), is_device));
  if (v) RET_IF(copy_out(h, v, h->v, h->ds.P * sizeof(float), is_device));
  if (step) { long long s = 0; RET_IF(copy_out(h, &s, h->step_dev, sizeof(s), 0)); *step = s; }
  return GNEP_OK;
}
int gnep_set_opt_state(gnep_handle *h, const float *m, const float *v, int64_t step, int is_device) {
  if (!h || step < 0) return fail(h, GNEP_EINVAL, "null handle or negative step");
  if (m) RET_IF(copy_in(h, h->m, m, h->ds.P * sizeof(float), is_device));
  if (v) RET_IF(copy_in(h, h->v, v, h->ds.P * sizeof(float), is_device));
  long long s = step;
  return copy_in(h, h->step_dev, &s, sizeof(s), 0);
}

int gnep_set_targets(gnep_handle *h, const double *E, const double *F, const double *W, int is_device) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  h->hasE = E != nullptr; h->hasF = F != nullptr; h->hasV = W != nullptr;
  if (E && h->S) RET_IF(copy_in(h, h->Eref, E, h->S * sizeof(double), is_device));
  if (W && h->S) RET_IF(copy_in(h, h->Wref, W, (size_t)h->S * 6 * sizeof(double), is_device));
  if (F && h->N) {
    double *tmp = nullptr;
    const double *src = F;
    if (!is_device) {
      CK(cudaMalloc((void **)&tmp, (size_t)h->N * 3 * sizeof(double)));
      cudaError_t e = cudaMemcpyAsync(tmp, F, (size_t)h->N * 3 * sizeof(double), cudaMemcpyHostToDevice, h->stream);
      if (e != cudaSuccess) { cudaFree(tmp); return fail(h, GNEP_ECUDA, cudaGetErrorString(e)); }
      src = tmp;
    }
    LAUNCH(h, k_permute_fref, cdiv(h->N, 256), 256, 0, h->N, h->perm, src, h->Fref_s);
    cudaError_t e = cudaStreamSynchronize(h->stream);
    if (tmp) cudaFree(tmp);
    if (e != cudaSuccess) return fail(h, GNEP_ECUDA, cudaGetErrorString(e));
  }
  if (h->graph) { cudaGraphExecDestroy(h->graph); h->graph = nullptr; }   // hasE/F/V are baked into the graph
  return GNEP_OK;
}

int gnep_set_weights(gnep_handle *h, const double *we, const double *wf, const double *wv, int is_device) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  const int S = h->S;
  std::vector<double> w((size_t)3 * S, 1.0);
  const double *src[3] = {we, wf, wv};
  for (int k = 0; k < 3; ++k)
    if (src[k] && S)
      CK(cudaMemcpy(w.data() + (size_t)k * S, src[k], (size_t)S * sizeof(double), is_device ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost));
  for (double x : w) if (!(x >= 0) || !std::isfinite(x)) return fail(h, GNEP_EINVAL, "weights must be finite and >= 0");
  double Z[3] = {0, 0, 0};
  for (int s = 0; s < S; ++s) {
    Z[0] += w[s]; Z[1] += w[(size_t)S + s] * (double)(h->host_aoff[s + 1] - h->host_aoff[s]); Z[2] += w[(size_t)2 * S + s];
  }
  for (int k = 0; k < 3; ++k) h->Zloc[k] = Z[k];
  if (S) RET_IF(copy_in(h, h->wgt, w.data(), w.size() * sizeof(double), 0));
  if (h->graph) { cudaGraphExecDestroy(h->graph); h->graph = nullptr; }   // the normalisers are kernel arguments of the graph
  return GNEP_OK;
}

int gnep_loss_norms(const gnep_handle *h, double *z) {
  if (!h || !z) return fail(h, GNEP_EINVAL, "null argument");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  for (int k = 0; k < 3; ++k) z[k] = h->Zloc[k];
  return GNEP_OK;
}

int gnep_load_batch(gnep_handle *h, int32_t S, const int32_t *aoff, const double *pos, const double *cells,
                    const int32_t *types, const double *Eref, const double *Fref, const double *Wref, int is_device) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (S < 0 || !aoff) return fail(h, GNEP_EINVAL, "bad n_structs / atom_offsets");
  if (aoff[0] != 0) return fail(h, GNEP_EINVAL, "atom_offsets[0] must be 0");
  for (int s = 0; s < S; ++s) if (aoff[s + 1] < aoff[s]) return fail(h, GNEP_EINVAL, "atom_offsets not ascending");
  const int N = aoff[S];
  if (N > 0 && (!pos || !cells || !types)) return fail(h, GNEP_EINVAL, "null positions / cells / types");
  CK(cudaStreamSynchronize(h->stream));
  free_batch(h);
  const DevSpec &d = h->ds;
  const int T = d.T;
  try {
    // ---- host copies of the small arrays ----
    std::vector<double> hcell((size_t)S * 9);
    std::vector<int> htype(N);
    if (S) CK(cudaMemcpy(hcell.data(), cells, hcell.size() * sizeof(double), is_device ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost));
    if (N) CK(cudaMemcpy(htype.data(), types, (size_t)N * sizeof(int), is_device ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost));
    for (int i = 0; i < N; ++i) if (htype[i] < 0 || htype[i] >= T) return fail(h, GNEP_ERANGE, "species id out of range");
    // ---- per-structure geometry and bins ----
    std::vector<StructGeo> geo(S);
    std::vector<int> struct_of(N);
    int total_bins = 0;
    const double rc = h->spec.rc_radial;
    for (int s = 0; s < S; ++s) {
      StructGeo &g = geo[s];
      double hh[3];
      memcpy(g.cell, &hcell[(size_t)s * 9], 9 * sizeof(double));
      if (cell_geometry(g.cell, g.inv, hh)) return fail(h, GNEP_ERANGE, "degenerate cell (zero volume)");
      for (int a = 0; a < 3; ++a) g.nb[a] = std::max(1, (int)std::floor(hh[a] / rc));
      while ((int64_t)g.nb[0] * g.nb[1] * g.nb[2] > 4096) {
        int big = g.nb[0] >= g.nb[1] && g.nb[0] >= g.nb[2] ? 0 : (g.nb[1] >= g.nb[2] ? 1 : 2);
        g.nb[big] = (g.nb[big] + 1) / 2;
      }
      for (int a = 0; a < 3; ++a) {
        g.m[a] = std::max(1, (int)std::ceil(rc * g.nb[a] / hh[a]));
        if (g.m[a] > 127) return fail(h, GNEP_ERANGE, "cell much smaller than the cutoff (more than 127 images per axis)");
      }
      g.bin_base = total_bins;
      total_bins += g.nb[0] * g.nb[1] * g.nb[2];
      g.a0 = aoff[s]; g.a1 = aoff[s + 1];
      for (int i = g.a0; i < g.a1; ++i) struct_of[i] = s;
    }
    // ---- species sort (stable) ----
    std::vector<int> perm(N), inv(N), type_s(N), struct_s(N);
    {
      std::vector<int> cnt(T + 1, 0);
      for (int i = 0; i < N; ++i) cnt[htype[i] + 1]++;
      for (int t = 0; t < T; ++t) cnt[t + 1] += cnt[t];
      for (int t = 0; t <= GNEP_MAX_SPECIES_C; ++t) h->sm.start[t] = cnt[std::min(t, T)];
      std::vector<int> cur(cnt.begin(), cnt.end() - 1);
      for (int i = 0; i < N; ++i) { int a = cur[htype[i]]++; perm[a] = i; inv[i] = a; }
      for (int a = 0; a < N; ++a) { type_s[a] = htype[perm[a]]; struct_s[a] = struct_of[perm[a]]; }
    }
    std::vector<int> srange((size_t)std::max(S, 1) * T * 2, 0);
    {
      std::vector<int> run(T);
      for (int t = 0; t < T; ++t) run[t] = h->sm.start[t];
      for (int s = 0; s < S; ++s) {
        std::vector<int> c(T, 0);
        for (int i = aoff[s]; i < aoff[s + 1]; ++i) c[htype[i]]++;
        for (int t = 0; t < T; ++t) { srange[((size_t)s * T + t) * 2] = run[t]; run[t] += c[t]; srange[((size_t)s * T + t) * 2 + 1] = run[t]; }
      }
    }
    h->N = N; h->S = S;
    // ---- device inputs ----
    double *d_pos_in = nullptr; bool own_pos = false;
    if (N) {
      if (is_device) d_pos_in = const_cast<double *>(pos);
      else { CK(cudaMalloc((void **)&d_pos_in, (size_t)N * 3 * sizeof(double))); own_pos = true;
             CK(cudaMemcpy(d_pos_in, pos, (size_t)N * 3 * sizeof(double), cudaMemcpyHostToDevice)); }
    }
    std::vector<void *> tmp;
    auto talloc = [&](void **p, size_t bytes) -> cudaError_t { cudaError_t e = cudaMalloc(p, std::max<size_t>(bytes, 16)); if (e == cudaSuccess) tmp.push_back(*p); return e; };
    auto tfree = [&]() { for (void *p : tmp) cudaFree(p); tmp.clear(); if (own_pos) { cudaFree(d_pos_in); own_pos = false; } };
#define CKT(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { tfree(); free_batch(h); return fail(h, e_ == cudaErrorMemoryAllocation ? GNEP_ENOMEM : GNEP_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); } } while (0)
    StructGeo *d_geo; int *d_struct_of, *d_type, *d_inv, *d_binid, *d_bin_count, *d_bin_start, *d_bin_cursor, *d_bin_atoms, *d_cntR, *d_cntA;
    double *d_wpos;
    CKT(talloc((void **)&d_geo, sizeof(StructGeo) * S)); CKT(talloc((void **)&d_struct_of, sizeof(int) * N));
    CKT(talloc((void **)&d_type, sizeof(int) * N)); CKT(talloc((void **)&d_inv, sizeof(int) * N));
    CKT(talloc((void **)&d_binid, sizeof(int) * N)); CKT(talloc((void **)&d_bin_count, sizeof(int) * (total_bins + 1)));
    CKT(talloc((void **)&d_bin_start, sizeof(int) * (total_bins + 1))); CKT(talloc((void **)&d_bin_cursor, sizeof(int) * (total_bins + 1)));
    CKT(talloc((void **)&d_bin_atoms, sizeof(int) * N)); CKT(talloc((void **)&d_cntR, sizeof(int) * N)); CKT(talloc((void **)&d_cntA, sizeof(int) * N));
    CKT(talloc((void **)&d_wpos, sizeof(double) * 3 * N));
    cudaStream_t st = h->stream;
    if (S) CKT(cudaMemcpyAsync(d_geo, geo.data(), sizeof(StructGeo) * S, cudaMemcpyHostToDevice, st));
    if (N) {
      CKT(cudaMemcpyAsync(d_struct_of, struct_of.data(), sizeof(int) * N, cudaMemcpyHostToDevice, st));
      CKT(cudaMemcpyAsync(d_type, htype.data(), sizeof(int) * N, cudaMemcpyHostToDevice, st));
      CKT(cudaMemcpyAsync(d_inv, inv.data(), sizeof(int) * N, cudaMemcpyHostToDevice, st));
    }
    CKT(cudaMemsetAsync(d_bin_count, 0, sizeof(int) * (total_bins + 1), st));
    CKT(cudaMemsetAsync(d_bin_cursor, 0, sizeof(int) * (total_bins + 1), st));
    const int gN = cdiv(N, 128);
    LAUNCH(h, k_wrap_bin, gN, 128, 0, N, d_struct_of, d_geo, d_pos_in, d_wpos, d_binid, d_bin_count);
    std::vector<int> bins(total_bins + 1, 0);
    CKT(cudaMemcpyAsync(bins.data(), d_bin_count, sizeof(int) * (total_bins + 1), cudaMemcpyDeviceToHost, st));
    CKT(cudaStreamSynchronize(st));
    { int run = 0; for (int b = 0; b <= total_bins; ++b) { int c = bins[b]; bins[b] = run; run += c; } }
    CKT(cudaMemcpyAsync(d_bin_start, bins.data(), sizeof(int) * (total_bins + 1), cudaMemcpyHostToDevice, st));
    LAUNCH(h, k_bin_fill, gN, 128, 0, N, d_binid, d_bin_start, d_bin_cursor, d_bin_atoms);
    const double rcR2 = h->spec.rc_radial * h->spec.rc_radial, rcA2 = h->spec.rc_angular * h->spec.rc_angular;
    LAUNCH(h, k_nbr_count, gN, 128, 0, N, d_struct_of, d_geo, d_wpos, d_binid, d_bin_start, d_bin_atoms, rcR2, rcA2, d_cntR, d_cntA);
    std::vector<int> cR(N), cA(N);
    if (N) {
      CKT(cudaMemcpyAsync(cR.data(), d_cntR, sizeof(int) * N, cudaMemcpyDeviceToHost, st));
      CKT(cudaMemcpyAsync(cA.data(), d_cntA, sizeof(int) * N, cudaMemcpyDeviceToHost, st));
    }
    CKT(cudaStreamSynchronize(st));
    std::vector<int64_t> rowR(N + 1, 0), rowA(N + 1, 0);
    for (int i = 0; i < N; ++i) { rowR[i + 1] = rowR[i] + cR[i]; rowA[i + 1] = rowA[i] + cA[i]; }
    const int64_t nR = rowR[N], nA = rowA[N];
    if (N >= (1 << 28)) { tfree(); free_batch(h); return fail(h, GNEP_ERANGE, "2^28 or more atoms"); }
    if (nR >= (int64_t)1 << 31) { tfree(); free_batch(h); return fail(h, GNEP_ERANGE, "2^31 or more radial pairs"); }
    std::vector<int> rowRs(N + 1, 0), rowAs(N + 1, 0);
    // radial rows start at even record indices (32-byte aligned): the walk reads two 16-byte records per 256-bit load
    for (int a = 0; a < N; ++a) { rowRs[a + 1] = rowRs[a] + ((cR[perm[a]] + 1) & ~1); rowAs[a + 1] = rowAs[a] + cA[perm[a]]; }
    h->nR = nR; h->nA = nA;
    // ---- persistent batch arrays ----
    int rc_;
#define BA(ptr, n) if ((rc_ = dalloc(h, &(ptr), (n), true)) != GNEP_OK) { tfree(); free_batch(h); return rc_; }
    BA(h->perm, N); BA(h->type_s, N); BA(h->struct_s, N); BA(h->segR, (size_t)N * (T + 1) + 1);
    BA(h->pairR, (size_t)rowRs[N] + 2);
    BA(h->exp_row[0], N + 1); BA(h->exp_row[1], N + 1); BA(h->exp_j[0], nR); BA(h->exp_sh[0], nR); BA(h->exp_j[1], nA); BA(h->exp_sh[1], nA);
    BA(h->srange, srange.size()); BA(h->Eref, S); BA(h->Wref, (size_t)S * 6); BA(h->Fref_s, (size_t)N * 3);
    BA(h->wgt, (size_t)3 * S);
    h->host_aoff.assign(aoff, aoff + S + 1);
    int *d_rowRs, *d_shA; unsigned long long *d_ekey; float *d_er;
    CKT(talloc((void **)&d_rowRs, sizeof(int) * (N + 1))); CKT(talloc((void **)&d_shA, sizeof(int) * nA));
    BA(h->rowAu, N + 1); BA(h->segAu, (size_t)N * (T + 1) + 1); BA(h->atomAu, nA); BA(h->pairAu, nA); BA(h->revAu, nA);
    int *d_rowAu = h->rowAu, *d_segAu = h->segAu, *d_atomAu = h->atomAu; float4 *d_pairAu = h->pairAu;
    CKT(talloc((void **)&d_ekey, sizeof(unsigned long long) * nR)); CKT(talloc((void **)&d_er, sizeof(float) * 3 * nR));
    CKT(cudaMemcpyAsync(h->exp_row[0], rowR.data(), sizeof(int64_t) * (N + 1), cudaMemcpyHostToDevice, st));
    CKT(cudaMemcpyAsync(h->exp_row[1], rowA.data(), sizeof(int64_t) * (N + 1), cudaMemcpyHostToDevice, st));
    CKT(cudaMemcpyAsync(d_rowRs, rowRs.data(), sizeof(int) * (N + 1), cudaMemcpyHostToDevice, st));
    CKT(cudaMemcpyAsync(d_rowAu, rowAs.data(), sizeof(int) * (N + 1), cudaMemcpyHostToDevice, st));
    if (N) {
      CKT(cudaMemcpyAsync(h->perm, perm.data(), sizeof(int) * N, cudaMemcpyHostToDevice, st));
      CKT(cudaMemcpyAsync(h->type_s, type_s.data(), sizeof(int) * N, cudaMemcpyHostToDevice, st));
      CKT(cudaMemcpyAsync(h->struct_s, struct_s.data(), sizeof(int) * N, cudaMemcpyHostToDevice, st));
    }
    CKT(cudaMemcpyAsync(h->srange, srange.data(), sizeof(int) * srange.size(), cudaMemcpyHostToDevice, st));
    // radial rows are padded to an even record count and the walk loads records in pairs: the pad slots (and the two
    // records past the last row) must hold a valid neighbour index for the one-ahead gather of k_radial_adj
    CKT(cudaMemsetAsync(h->pairR, 0, sizeof(float4) * ((size_t)rowRs[N] + 2), st));
    LAUNCH(h, k_nbr_fill, gN, 128, 0, N, d_struct_of, d_geo, d_wpos, d_binid, d_bin_start, d_bin_atoms, rcR2, rcA2, h->exp_row[0], d_ekey, d_er);
    LAUNCH(h, k_nbr_scatter, cdiv((int64_t)N * 32, 256), 256, 0, N, T, d_struct_of, d_geo, d_type, d_inv, h->exp_row[0], h->exp_row[1], d_rowRs,
           d_rowAu, d_ekey, d_er, h->exp_j[0], h->exp_sh[0], h->exp_j[1], h->exp_sh[1], h->pairR, d_pairAu, d_shA, h->segR, d_segAu, d_atomAu);
    CKT(cudaGetLastError());
    std::vector<int> segAu((size_t)N * (T + 1) + 1, 0);
    if (N) CKT(cudaMemcpyAsync(segAu.data(), d_segAu, sizeof(int) * (size_t)N * (T + 1), cudaMemcpyDeviceToHost, st));
    CKT(cudaStreamSynchronize(st));
    // ---- tiles of the angular moment kernels: 32 atoms of one central species, atoms sorted by their per-species
    // neighbour counts (descending), so that the rows a warp walks in lock step have equal lengths; the last tile of a
    // species is filled up with -1 (idle lanes)
    std::vector<int> tiles;
    if (h->tile_path) {
      std::vector<std::pair<uint64_t, int>> keyed;
      for (int t = 0; t < T; ++t) {
        const int a0 = h->sm.start[t], a1 = h->sm.start[t + 1];
        keyed.clear();
        for (int a = a0; a < a1; ++a) {
          uint64_t key = 0;
          for (int J = 0; J < T; ++J)
            key = (key << 16) | (uint64_t)std::min(segAu[(size_t)a * (T + 1) + J + 1] - segAu[(size_t)a * (T + 1) + J], 65535);
          keyed.emplace_back(~key, a);               // descending counts, ascending atom index among equals
        }
        std::sort(keyed.begin(), keyed.end());
        for (auto &kv : keyed) tiles.push_back(kv.second);
        while (tiles.size() % ANG_TILE) tiles.push_back(-1);
      }
    }
    h->n_tilesA = (int)(tiles.size() / ANG_TILE);
    BA(h->tilesA, tiles.size());
    if (!tiles.empty()) CKT(cudaMemcpyAsync(h->tilesA, tiles.data(), sizeof(int) * tiles.size(), cudaMemcpyHostToDevice, st));
    // ---- warp-tile path: the angular list once more with every (atom, J) segment padded to a multiple of 4 pairs by
    // zero-contribution dummies (k_pad_angular), so that the 4-pair register tiles of the sweeps never straddle a segment
    std::vector<int> segAp;
    if (!h->tile_path) {
      segAp.assign((size_t)N * (T + 1) + 1, 0);
      int64_t nAp = 0;
      for (int a = 0; a < N; ++a) {
        for (int J = 0; J < T; ++J) {
          segAp[(size_t)a * (T + 1) + J] = (int)nAp;
          nAp += (segAu[(size_t)a * (T + 1) + J + 1] - segAu[(size_t)a * (T + 1) + J] + 3) / 4 * 4;
        }
        segAp[(size_t)a * (T + 1) + T] = (int)nAp;
      }
      if (nAp >= (int64_t)1 << 31) { tfree(); free_batch(h); return fail(h, GNEP_ERANGE, "2^31 or more (padded) angular pairs"); }
      BA(h->segA, (size_t)N * (T + 1) + 1); BA(h->atomA, nAp); BA(h->pairA, nAp);
      CKT(cudaMemcpyAsync(h->segA, segAp.data(), sizeof(int) * ((size_t)N * (T + 1) + 1), cudaMemcpyHostToDevice, st));
      LAUNCH(h, k_pad_angular, cdiv((int64_t)N * 32, 256), 256, 0, N, T, d_segAu, h->segA, d_pairAu, h->pairA, h->atomA,
             (float)(2.0 * h->spec.rc_angular));
    }
    LAUNCH(h, k_nbr_reverse, cdiv((int64_t)N * 32, 256), 256, 0, N, h->rowAu, h->pairAu, d_shA, h->revAu);
    CKT(cudaGetLastError());
    CKT(cudaStreamSynchronize(st));
    tfree();
    // ---- work decomposition of the network / gradient kernels ----
    // (small batches -- see below -- run the network on plain FMAs, one warp per atom, with short atom ranges per CTA)
    bool small = N < 2 * h->num_sms * RAD_THREADS;
    if (const char *e = getenv("GNEP_SMALL_BATCH")) small = atoi(e) != 0;
    h->net_small = small && d.Nn <= 128 && d.Ndes <= 128 && sizeof(float) * net_small_bwd_floats(d) <= 200 * 1024 &&
                   sizeof(float) * net_small_fwd_floats(d) <= 200 * 1024;
    int tiles_total = 0;
    for (int t = 0; t < T; ++t) tiles_total += cdiv(h->sm.start[t + 1] - h->sm.start[t], 128);
    h->sm.cta_base[0] = 0; h->sm.chunk_base[0] = 0; h->sm.gw_base[0] = 0;
    for (int t = 0; t < GNEP_MAX_SPECIES_C; ++t) {
      int nt = t < T ? h->sm.start[t + 1] - h->sm.start[t] : 0;
      // k_net_tc: persistent CTAs (two 128-atom tiles in flight each), shared out by tile count
      int tiles = cdiv(nt, 128);
      int nc = tiles > 0 ? std::max(1, std::min(cdiv(tiles, 2), (int)((double)h->num_sms * tiles / std::max(tiles_total, 1) + 0.5))) : 0;
      h->sm.cta_base[t + 1] = h->sm.cta_base[t] + nc;
      // k_cgrad_radial: K-chunks
      int want = nt > 0 ? std::max(1, std::min(cdiv(nt, 32), (int)((4.0 * h->num_sms * nt) / std::max(N, 1) + 0.5))) : 0;
      int ca = want > 0 ? ((cdiv(nt, want) + 31) / 32) * 32 : 32;
      h->sm.chunk_atoms[t] = ca;
      h->sm.chunk_base[t + 1] = h->sm.chunk_base[t] + (nt > 0 ? cdiv(nt, ca) : 0);
      // k_gradw_tc: one contiguous atom range per CTA
      int gwant = nt > 0 ? std::max(1, std::min(cdiv(nt, 4 * GW_KS), (int)((double)h->num_sms * nt / std::max(N, 1) + 0.5))) : 0;
      int ga = gwant > 0 ? pad_to(cdiv(nt, gwant), GW_KS) : GW_KS;
      if (h->net_small) ga = NS_ATOMS;             // k_net_small_fwd / bwd: short contiguous atom ranges of one species
      h->sm.gw_atoms[t] = ga;
      h->sm.gw_base[t + 1] = h->sm.gw_base[t] + (nt > 0 ? cdiv(nt, ga) : 0);
    }
    if (h->net_small)   // the radial c-gradient partials come from k_net_small_bwd: one row per CTA of that kernel
      for (int t = 0; t <= GNEP_MAX_SPECIES_C; ++t) h->sm.chunk_base[t] = h->sm.gw_base[t];
    h->n_cta_net = h->sm.cta_base[GNEP_MAX_SPECIES_C];
    h->n_chunks = h->sm.chunk_base[GNEP_MAX_SPECIES_C];
    h->n_gw = h->sm.gw_base[GNEP_MAX_SPECIES_C];
    if (h->tile_path) {
      h->grid_adj = std::min(h->n_tilesA, h->occ_adj * h->num_sms);
      h->grid_cg = std::min(h->n_tilesA, h->occ_cg * h->num_sms);
    } else {   // only k_angw_cgrad keeps accumulators: persistent warps, four CTAs per SM
      h->grid_adj = 0;
      h->grid_cg = std::max(1, std::min(cdiv(N, ANG_WARPS), 4 * h->num_sms));
    }
    // A mini-batch of a few hundred atoms (the paper trains with batch size 1) cannot fill the SMs with the
    // large-batch mappings (one thread per atom in the radial sweeps, ANG_TA atoms per warp in the angular ones): below
    // two CTAs per SM of the radial kernels the atom tiles shrink until there are about four CTAs per SM and the radial
    // force / adjoint sweeps use RAD_SPLIT lanes per atom.  GNEP_SMALL_BATCH=0/1 forces either set (tests run both).
    h->ta_ang = small ? std::max(1, std::min(ANG_TA, cdiv(N, 4 * h->num_sms * ANG_WARPS))) : ANG_TA;
    h->ta_frc = small ? std::max(1, std::min(FRC_TA, cdiv(N, 5 * h->num_sms * FRC_WARPS))) : FRC_TA;
    h->rad_split = small;
    h->rad_lanes = (int64_t)N * RAD_SPLIT_WIDE <= (int64_t)4 * h->num_sms * RAD_THREADS ? RAD_SPLIT_WIDE : RAD_SPLIT;
    for (int t = 0; t <= GNEP_MAX_SPECIES_C; ++t) { h->rm.chunk_base[t] = h->sm.chunk_base[t]; h->rm.gw_base[t] = h->sm.gw_base[t]; }
    const int ca_warps = h->tile_path ? ang_warps(d) : ANG_WARPS;
    h->rm.n_warps_ca = N > 0 ? (h->grid_adj + h->grid_cg) * ca_warps : 0;   // partial rows: the beta half (adjoint sweep) then the alpha half
    // ---- per-atom state ----
    const size_t n = N;
    const size_t npad = n + GW_PAD_ROWS;
    const size_t nxt = (npad + 127) / 128 * 128;   // x, p: whole 128-atom blocks of the XT layout (net_tc_kernels.cuh)   // k_gradw_tc bulk-copies whole windows of rows: zeroed rows past the end
    BA(h->q, npad * d.Ndes); BA(h->Sn, n * d.NA * d.nlmS); BA(h->x, nxt * d.NnS); BA(h->Ei, n); BA(h->Ep, n * d.Ndes);
    BA(h->etil, n * T * d.KRp); BA(h->M1, n * T * d.KRp); BA(h->M2, n * T * d.KRp); BA(h->D, npad * d.Ndes); BA(h->Tn, n * d.NA * d.nlmS); if (h->tile_path) BA(h->Beta, n * d.NA * d.nlmS);   /* (read by the slot-group adjoint sweep only) */ BA(h->A1, h->tile_path ? n * ang_groups(d.L) * T * d.KAp * ANG_GS : n * T * d.KAp * ANGW_NLM);
    if (!h->tile_path) BA(h->A2, n * T * d.KAp * ANGW_NLM);
    BA(h->gbar, n * d.Ndes); BA(h->pbuf, nxt * d.NnS); BA(h->eat, npad); BA(h->Wat, n * 6);
    BA(h->Fat, n); BA(h->fpair, h->nA); BA(h->u, n);
    BA(h->Es, S); BA(h->Ws, (size_t)S * 6); BA(h->parts, (size_t)S * 3 + LOSS_T2_CTAS); BA(h->e_s, S); BA(h->omega, (size_t)S * 6);
    BA(h->partialCR, (size_t)std::max(h->n_chunks, 1) * d.NR * T * d.KRp);
    BA(h->partialCA, (size_t)std::max(h->rm.n_warps_ca, 1) * T * T * d.NA * d.KAp);
    BA(h->partialW, (size_t)std::max(h->n_gw, 1) * d.Nn * d.Ndes);
    BA(h->partialB, (size_t)std::max(h->n_gw, 1) * (2 * d.Nn + 1));
    // slots of the (l,m) rows that no slot group of this model writes (l_max < 4) are read as zeros
    CKT(cudaMemsetAsync(h->Sn, 0, sizeof(float) * n * d.NA * d.nlmS, st));
    CKT(cudaMemsetAsync(h->Tn, 0, sizeof(float) * n * d.NA * d.nlmS, st));
    CKT(cudaMemsetAsync(h->q + n * d.Ndes, 0, sizeof(float) * GW_PAD_ROWS * d.Ndes, st));
    CKT(cudaMemsetAsync(h->D + n * d.Ndes, 0, sizeof(float) * GW_PAD_ROWS * d.Ndes, st));
    CKT(cudaMemsetAsync(h->x, 0, sizeof(float) * nxt * d.NnS, st));
    CKT(cudaMemsetAsync(h->pbuf, 0, sizeof(float) * nxt * d.NnS, st));
    CKT(cudaMemsetAsync(h->eat + n, 0, sizeof(float) * GW_PAD_ROWS, st));
#undef BA
#undef CKT
    h->loaded = true;
    if (N > 0) { RET_IF(enqueue_geometry_moments(h)); RET_IF(check_launch(h)); }
    RET_IF(gnep_set_weights(h, nullptr, nullptr, nullptr, 0));
    return gnep_set_targets(h, Eref, Fref, Wref, is_device);
  } catch (const std::bad_alloc &) {
    free_batch(h);
    return fail(h, GNEP_ENOMEM, "out of host memory");
  }
}

int gnep_batch_info(const gnep_handle *h, int64_t *n_atoms, int64_t *n_structs, int64_t *nR, int64_t *nA) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  if (n_atoms) *n_atoms = h->N;
  if (n_structs) *n_structs = h->S;
  if (nR) *nR = h->nR;
  if (nA) *nA = h->nA;
  return GNEP_OK;
}

int gnep_neighbor_list(const gnep_handle *h, int which, int64_t *n_pairs, int64_t *row_ptr, int32_t *j, int8_t *shift3,
                       int64_t capacity, int is_device) {
  if (!h || (which != 0 && which != 1)) return fail(h, GNEP_EINVAL, "bad argument");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  const int64_t np = which == 0 ? h->nR : h->nA;
  if (n_pairs) *n_pairs = np;
  if ((j || shift3) && capacity < np) return fail(h, GNEP_EINVAL, "capacity smaller than the pair count");
  if (row_ptr) RET_IF(copy_out(h, row_ptr, h->exp_row[which], (size_t)(h->N + 1) * sizeof(int64_t), is_device));
  if (j && np) RET_IF(copy_out(h, j, h->exp_j[which], (size_t)np * sizeof(int32_t), is_device));
  if (shift3 && np) {
    std::vector<int> packed(np);
    RET_IF(copy_out(h, packed.data(), h->exp_sh[which], (size_t)np * sizeof(int), 0));
    std::vector<int8_t> sh((size_t)np * 3);
    for (int64_t p = 0; p < np; ++p) {
      sh[3 * p] = (int8_t)(((packed[p] >> 16) & 255) - 128);
      sh[3 * p + 1] = (int8_t)(((packed[p] >> 8) & 255) - 128);
      sh[3 * p + 2] = (int8_t)((packed[p] & 255) - 128);
    }
    if (is_device) { gnep_handle *hh = const_cast<gnep_handle *>(h); return copy_in(hh, shift3, sh.data(), sh.size(), 0); }
    memcpy(shift3, sh.data(), sh.size());
  }
  return GNEP_OK;
}

int gnep_descriptors(gnep_handle *h, float *q, int is_device) {
  if (!h || !q) return fail(h, GNEP_EINVAL, "null argument");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  if (h->N == 0) return GNEP_OK;
  RET_IF(enqueue_descriptors(h));
  const size_t n = (size_t)h->N * h->ds.Ndes;
  float *dst = q; float *tmp = nullptr;
  if (!is_device) { CK(cudaMalloc((void **)&tmp, n * sizeof(float))); dst = tmp; }
  LAUNCH(h, k_unpermute_rows, cdiv(n, 256), 256, 0, h->N, h->ds.Ndes, h->perm, h->q, dst);
  int rc = check_launch(h);
  if (rc == GNEP_OK && tmp) rc = copy_out(h, q, tmp, n * sizeof(float), 0);
  else if (rc == GNEP_OK) { cudaError_t e = cudaStreamSynchronize(h->stream); if (e != cudaSuccess) rc = fail(h, GNEP_ECUDA, cudaGetErrorString(e)); }
  if (tmp) cudaFree(tmp);
  return rc;
}

int gnep_predict(gnep_handle *h, float *energy, float *force, float *virial, int is_device) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  if (h->N > 0 || h->S > 0) { RET_IF(enqueue_forward(h)); RET_IF(check_launch(h)); }
  std::vector<void *> tmp;
  auto run = [&]() -> int {
    if (energy && h->S) {
      float *dst = energy;
      if (!is_device) { CK(cudaMalloc((void **)&dst, h->S * sizeof(float))); tmp.push_back(dst); }
      LAUNCH(h, k_d2f, cdiv(h->S, 256), 256, 0, h->S, h->Es, dst);
      if (!is_device) RET_IF(copy_out(h, energy, dst, h->S * sizeof(float), 0));
    }
    if (virial && h->S) {
      float *dst = virial;
      if (!is_device) { CK(cudaMalloc((void **)&dst, (size_t)h->S * 6 * sizeof(float))); tmp.push_back(dst); }
      LAUNCH(h, k_d2f, cdiv(h->S * 6, 256), 256, 0, h->S * 6, h->Ws, dst);
      if (!is_device) RET_IF(copy_out(h, virial, dst, (size_t)h->S * 6 * sizeof(float), 0));
    }
    if (force && h->N) {
      float *dst = force;
      if (!is_device) { CK(cudaMalloc((void **)&dst, (size_t)h->N * 3 * sizeof(float))); tmp.push_back(dst); }
      LAUNCH(h, k_unpermute_force, cdiv(h->N, 256), 256, 0, h->N, h->perm, h->Fat, dst);
      if (!is_device) RET_IF(copy_out(h, force, dst, (size_t)h->N * 3 * sizeof(float), 0));
    }
    RET_IF(check_launch(h));
    CK(cudaStreamSynchronize(h->stream));
    return GNEP_OK;
  };
  int rc = run();
  for (void *p : tmp) cudaFree(p);
  return rc;
}

int gnep_loss_and_grad(gnep_handle *h, float *loss_terms, float *grad, int is_device) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  prof_begin(h);
  RET_IF(enqueue_forward(h));
  RET_IF(enqueue_backward(h));
  RET_IF(check_launch(h));
  if (grad) RET_IF(copy_out(h, grad, h->grad, h->ds.P * sizeof(float), is_device));
  if (loss_terms) RET_IF(fetch_terms(h, loss_terms));
  return GNEP_OK;
}

int gnep_evaluate(gnep_handle *h, float *rmse) {
  if (!h || !rmse) return fail(h, GNEP_EINVAL, "null argument");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  float t[5] = {0, 0, 0, 0, 0};
  if (h->N > 0 || h->S > 0) {
    h->eval_local = true;
    int rc = enqueue_forward(h);
    h->eval_local = false;
    RET_IF(rc);
    RET_IF(check_launch(h));
    RET_IF(fetch_terms(h, t));
  }
  for (int i = 0; i < 3; ++i) rmse[i] = std::sqrt(std::max(t[1 + i], 0.f));   // t_e, t_f, t_v are the mean squares of Eq.10-12
  return GNEP_OK;
}

int gnep_adam_step(gnep_handle *h, float lr, float beta1, float beta2, float eps) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (!(beta1 >= 0 && beta1 < 1 && beta2 >= 0 && beta2 < 1) || !(eps >= 0)) return fail(h, GNEP_EINVAL, "bad Adam constants");
  if (h->g_lr != lr) { set_lr(h, lr); h->g_lr = lr; }
  RET_IF(enqueue_adam(h, beta1, beta2, eps));
  return check_launch(h);
}

int gnep_train_epochs(gnep_handle *h, int32_t n_epochs, float lr, float beta1, float beta2, float eps, float *loss_terms) {
  if (!h || n_epochs < 0) return fail(h, GNEP_EINVAL, "bad argument");
  if (!h->loaded) return fail(h, GNEP_ESTATE, "no batch loaded");
  if (!(beta1 >= 0 && beta1 < 1 && beta2 >= 0 && beta2 < 1) || !(eps >= 0)) return fail(h, GNEP_EINVAL, "bad Adam constants");
  if (h->graph && (h->g_b1 != beta1 || h->g_b2 != beta2 || h->g_eps != eps)) {
    cudaGraphExecDestroy(h->graph); h->graph = nullptr;
  }
  if (!h->graph) {
    bool prof = h->prof; h->prof = false;
    int64_t before = h->launches;
    cudaGraph_t g = nullptr;
    CK(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
    h->fuse_adam = true; h->fuse_b1 = beta1; h->fuse_b2 = beta2; h->fuse_eps = eps;   // a9 inside a4 / a8 (reduce_kernels.cuh)
    int rc = enqueue_forward(h);
    if (rc == GNEP_OK) rc = enqueue_backward(h);
    h->fuse_adam = false;
    cudaError_t e = cudaStreamEndCapture(h->stream, &g);
    h->prof = prof;
    h->graph_launches = h->launches - before;
    h->launches = before;
    if (rc != GNEP_OK) { if (g) cudaGraphDestroy(g); return rc; }
    if (e != cudaSuccess) return fail(h, GNEP_ECUDA, std::string("graph capture: ") + cudaGetErrorString(e));
    e = cudaGraphInstantiate(&h->graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { h->graph = nullptr; return fail(h, GNEP_ECUDA, std::string("graph instantiate: ") + cudaGetErrorString(e)); }
    h->g_lr = -1.f; h->g_b1 = beta1; h->g_b2 = beta2; h->g_eps = eps;
  }
  if (h->g_lr != lr) { set_lr(h, lr); h->g_lr = lr; }   // outside the graph: a schedule only rewrites the device scalar
  for (int i = 0; i < n_epochs; ++i) { CK(cudaGraphLaunch(h->graph, h->stream)); h->launches += h->graph_launches; }
  if (loss_terms) RET_IF(fetch_terms(h, loss_terms));
  return GNEP_OK;
}

int gnep_set_global_norms(gnep_handle *h, const double *z, double l2_share) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (!z || z[0] < 0 || z[1] < 0 || z[2] < 0) { h->Zjob[0] = h->Zjob[1] = h->Zjob[2] = -1; h->l2_share = 1.0; }
  else {
    if (h->ds.loss_mode != 0) return fail(h, GNEP_EINVAL, "sharded normalisation needs loss_mode 0 (RMSE mode needs the global terms before the seeds)");
    if (!(l2_share >= 0 && l2_share <= 1)) return fail(h, GNEP_EINVAL, "l2_share must be in [0,1]");
    for (int k = 0; k < 3; ++k) h->Zjob[k] = z[k];
    h->l2_share = l2_share;
  }
  if (h->graph) { cudaGraphExecDestroy(h->graph); h->graph = nullptr; }
  return GNEP_OK;
}

int gnep_set_global_norm(gnep_handle *h, int64_t n_atoms_global, int64_t n_structs_global, double l2_share) {
  if (n_atoms_global < 0 || n_structs_global < 0) return gnep_set_global_norms(h, nullptr, 1.0);
  const double z[3] = {(double)n_structs_global, (double)n_atoms_global, (double)n_structs_global};
  return gnep_set_global_norms(h, z, l2_share);
}

int gnep_set_grad(gnep_handle *h, const float *grad, int is_device) {
  if (!h || !grad) return fail(h, GNEP_EINVAL, "null argument");
  return copy_in(h, h->grad, grad, h->ds.P * sizeof(float), is_device);
}

int gnep_measure_fp32_peak(gnep_handle *h, double min_ms, double *tflops, double *ms_out, double *sm_mhz) {
  if (!h || !tflops) return fail(h, GNEP_EINVAL, "null argument");
  if (!(min_ms > 0) || min_ms > 2000) return fail(h, GNEP_EINVAL, "min_ms must be in (0, 2000]");
  const int grid = h->num_sms * 8, block = 256;     // 2048 resident threads per SM
  float *sink = nullptr;
  CK(cudaMalloc((void **)&sink, sizeof(float) * (size_t)grid * block));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  auto run = [&](int iters, float *ms) -> cudaError_t {
    cudaEventRecord(e0, h->stream);
    k_ffma_peak<<<grid, block, 0, h->stream>>>(iters, 0.999f, 1e-3f, sink);
    h->launches++;
    cudaEventRecord(e1, h->stream);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, e0, e1);
    return e;
  };
  float ms = 0.f;
  int iters = 4096;
  cudaError_t e = run(iters, &ms);                  // warm-up and calibration
  if (e == cudaSuccess) {
    const double want = min_ms / std::max((double)ms, 1e-3) * iters;
    iters = (int)std::min(std::max(want, 4096.0), 2.0e8);
    e = run(iters, &ms);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(sink);
  if (e != cudaSuccess) return fail(h, GNEP_ECUDA, std::string("fp32 peak measurement: ") + cudaGetErrorString(e));
  const double flops = 2.0 * PEAK_CHAINS * PEAK_UNROLL * (double)iters * (double)grid * block;
  *tflops = flops / (ms * 1e-3) / 1e12;
  if (ms_out) *ms_out = ms;
  if (sm_mhz) *sm_mhz = *tflops * 1e12 / (2.0 * 128.0 * h->num_sms) / 1e6;   // the clock this rate implies at 128 lanes / SM
  return GNEP_OK;
}

int gnep_loss_terms_noalloc(gnep_handle *h, int32_t n_structs, const int32_t *atom_offsets, const float *energy,
                            const float *force, const float *virial, const double *Eref, const double *Fref,
                            const double *Wref, float *terms) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  if (n_structs < 1) return fail(h, GNEP_EINVAL, "n_structs must be at least 1");
  if (n_structs > NOALLOC_MAX_STRUCTS)
    return fail(h, GNEP_ERANGE, "gnep_loss_terms_noalloc: " + std::to_string(n_structs) + " structures exceed the fixed scratch of " +
                                    std::to_string(NOALLOC_MAX_STRUCTS) + " (split the batch, or use gnep_set_targets + gnep_loss_and_grad)");
  if (!atom_offsets || !terms) return fail(h, GNEP_EINVAL, "null atom_offsets / terms");
  if ((Eref && !energy) || (Fref && !force) || (Wref && !virial)) return fail(h, GNEP_EINVAL, "a reference without its prediction");
  double *scratch = nullptr;
  CK(noalloc_scratch(h->device, &scratch));
  // the array keeps the last call's contents: the partial sums are all rewritten, the ticket must start at zero
  CK(cudaMemsetAsync(scratch + 3 * NOALLOC_MAX_STRUCTS, 0, sizeof(unsigned), h->stream));
  NoAllocLoss lc;
  lc.S = n_structs; lc.loss_mode = h->ds.loss_mode;
  lc.lam_e = Eref ? h->spec.lambda_e : 0.0; lc.lam_f = Fref ? h->spec.lambda_f : 0.0; lc.lam_v = Wref ? h->spec.lambda_v : 0.0;
  LAUNCH(h, k_loss_terms_noalloc, n_structs, 128, 0, lc, atom_offsets, energy, force, virial, Eref, Fref, Wref, scratch, terms);
  return check_launch(h);
}

int gnep_launch_count(const gnep_handle *h, int64_t *n) {
  if (!h || !n) return fail(h, GNEP_EINVAL, "null argument");
  *n = h->launches;
  return GNEP_OK;
}

int gnep_set_profiling(gnep_handle *h, int on) {
  if (!h) return fail(h, GNEP_EINVAL, "null handle");
  h->prof = on != 0;
  return GNEP_OK;
}
int gnep_phase_times(const gnep_handle *h, const char **names, float *ms, int32_t capacity, int32_t *n) {
  if (!h || !n) return fail(h, GNEP_EINVAL, "null argument");
  gnep_handle *hh = const_cast<gnep_handle *>(h);
  if (hh->prof && !hh->phases.empty()) prof_collect(hh);
  *n = (int32_t)h->phase_ms.size();
  for (int i = 0; i < *n && i < capacity; ++i) { if (names) names[i] = h->phase_names[i]; if (ms) ms[i] = h->phase_ms[i]; }
  return GNEP_OK;
}

}  // extern "C"
