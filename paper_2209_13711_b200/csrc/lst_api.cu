// lst_api.cu -- the C-ABI of include/lst.h: context, module-map builder (host), workspace layout,
// event upload, the launch chain (optionally one CUDA graph per slot) and result views.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/lst.h"
#include "../../include/lst_test.h"
#include "lst_launch.h"

using namespace lst;

// ------------------------------------------------------------------ status text
static thread_local char g_cuda_err[256] = "no CUDA error recorded";
static thread_local char g_cap_err[640] = "workspace too small or object capacity exceeded";
static thread_local char g_inval_err[192] = "invalid argument";

static int cuda_fail(cudaError_t e, const char *where) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "CUDA error at %s: %s", where, cudaGetErrorString(e));
  return LST_ECUDA;
}
static int einval() {
  snprintf(g_inval_err, sizeof(g_inval_err), "invalid argument");
  return LST_EINVAL;
}
#define CU(call)                                          \
  do {                                                    \
    cudaError_t e_ = (call);                              \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);   \
  } while (0)

extern "C" const char *lst_strerror(int status) {
  switch (status) {
    case LST_OK: return "ok";
    case LST_EINVAL: return g_inval_err;
    case LST_ENOMEM: return g_cap_err;
    case LST_ECUDA: return g_cuda_err;
    case LST_ESTATE: return "call order violated";
    default: return "unknown status";
  }
}

// ------------------------------------------------------------------ config
extern "C" void lst_default_config(lst_config *c) {
  if (!c) return;
  memset(c, 0, sizeof(*c));
  const double s12 = std::sqrt(12.0);
  c->kB = 0.00299792458 * 3.8;
  c->pt_min = 0.8;
  c->n_sigma = 4.0;
  c->z0max = 15.0;
  c->d0max = 2.5;
  c->chi2max = 18.42;
  c->dr2max = 1e-4;
  c->map_kscale = 1.25;
  c->map_z0 = 20.0;
  c->ec_md_sys = 0.3;
  c->modez_slack = 0.15;
  c->seed_sig_phi = 0.001;
  c->seed_sig_pt = 0.01;
  c->seed_sig_z = 0.05;
  const double pitch_t[4] = {0.01, 0.009, 0.01, 0.009};
  const double len_z[4] = {0.15, 5.0, 0.0, 0.0}, len_r[4] = {0.0, 0.0, 0.15, 5.0};
  for (int k = 0; k < 4; ++k) {
    c->sig_t[k] = pitch_t[k] / s12;
    c->sig_z[k] = len_z[k] / s12;
    c->sig_r[k] = len_r[k] / s12;
  }
  c->dup_t5_shared = 5;
  c->dup_pt5_shared = 5;
  c->dup_pt3_shared = 3;
  c->s0_enabled = 1;
  c->start_layer_mask = 0x3u | (0x3u << 6) | (0x3u << 11);
  c->cap_md_per_hit = 1.0f;
  c->cap_ls_per_hit = 6.0f;
  c->cap_t3_per_hit = 6.0f;
  c->cap_t5_per_hit = 2.0f;
  c->cap_pt3_per_seed = 96.0f;
  c->cap_pt5_per_seed = 48.0f;
  c->cap_mdcand_per_hit = 64.0f;
  c->cap_lscand_per_hit = 512.0f;
  c->cap_t3cand_per_hit = 64.0f;
  c->cap_t5cand_per_hit = 16.0f;
  c->use_cuda_graph = 1;
  c->enum_pruning = 3;
  c->use_pdl = 1;
  c->batch_events = 1;
  /* trunc_cap: all 0 (no occupancy truncation); store_half: 0 */
}

static void make_params(const lst_config &c, Params *p) {
  memset(p, 0, sizeof(*p));
  p->kmax = c.kB / (2.0 * c.pt_min);
  p->kB = c.kB; p->ns = c.n_sigma; p->z0max = c.z0max; p->d0max = c.d0max; p->chi2max = c.chi2max;
  p->dr2max = c.dr2max; p->ec_md_sys = c.ec_md_sys; p->modez_slack = c.modez_slack;
  p->seed_sig_phi = c.seed_sig_phi; p->seed_sig_pt = c.seed_sig_pt; p->seed_sig_z = c.seed_sig_z;
  for (int k = 0; k < 4; ++k) {
    p->sig_t[k] = c.sig_t[k]; p->sig_z[k] = c.sig_z[k]; p->sig_r[k] = c.sig_r[k];
    p->f_sig_t[k] = (float)c.sig_t[k]; p->f_sig_z[k] = (float)c.sig_z[k]; p->f_sig_r[k] = (float)c.sig_r[k];
  }
  p->f_kmax = (float)p->kmax; p->f_ns = (float)c.n_sigma; p->f_z0max = (float)c.z0max;
  p->f_ec_md_sys = (float)c.ec_md_sys; p->f_modez_slack = (float)c.modez_slack;
  p->dup_t5 = c.dup_t5_shared; p->dup_pt5 = c.dup_pt5_shared; p->dup_pt3 = c.dup_pt3_shared;
  p->s0_enabled = c.s0_enabled;
  p->start_mask = c.start_layer_mask;
  for (int l = 0; l < 6; ++l) for (int k = 0; k < 16; ++k) p->trunc[l][k] = c.trunc_cap[l][k];
  // bin width >= 1.25 sqrt(dr2max): two seeds closer than sqrt(dr2max) in eta are in adjacent bins
  const double sq = std::sqrt(std::max(c.dr2max, 0.0));
  const double width = std::max(1.25 * sq, 8.0 / kEtaBins);
  p->eta_bin_inv = 1.0 / width;
  p->eta_nbins = std::min<int>(kEtaBins, (int)std::ceil(8.0 / width));
  p->dr_eta_pre = 1.001 * sq + 1e-12;
}

static bool geometry_ok(const lst_geometry *g) {
  if (!g || g->n_modules == 0 || !g->category || !g->logical_layer || !g->rmin || !g->rmax || !g->phic ||
      !g->half_phi || !g->zmin || !g->zmax)
    return false;
  for (uint32_t m = 0; m < g->n_modules; ++m) {
    if (g->category[m] > 3 || g->logical_layer[m] > 15) return false;
    // a sane box: 0 < rmin <= rmax, zmin <= zmax (equal for an endcap module: the sensor plane, and not
    // through z = 0), 0 < half_phi <= 0.6 rad (the azimuthal windows assume a module is narrow)
    if (!(g->rmin[m] > 0.0f) || !(g->rmax[m] >= g->rmin[m]) || !(g->zmax[m] >= g->zmin[m])) return false;
    if (!(g->half_phi[m] > 0.0f) || !(g->half_phi[m] <= 0.6f) || !(std::fabs(g->phic[m]) <= 6.3f)) return false;
    if (g->category[m] >= 2 && (g->zmin[m] != g->zmax[m] || g->zmin[m] == 0.0f)) return false;
    if (!(std::fabs(g->zmin[m]) <= 1e6f) || !(g->rmax[m] <= 1e6f)) return false;
  }
  return true;
}

// ------------------------------------------------------------------ C2 module map (host)
// PAPER.md:53-55 (Fig. 4).  Reading C2: B is connected to A iff B sits in a layer that may follow
// A's, and the phi and r-z intervals swept from A's box by helices with |kappa| <= kscale*kmax,
// |z0| <= map_z0 (and a d0max allowance in phi) overlap B's box.
namespace {
struct Box { double rlo, rhi, phi, hphi, zlo, zhi; bool endcap; };

inline void followers(int layer, int out[3], int *n) {
  *n = 0;
  if (layer < 6) {
    if (layer < 5) out[(*n)++] = layer + 1;
    out[(*n)++] = 6;
    out[(*n)++] = 11;
  } else if (layer != 10 && layer != 15) {
    out[(*n)++] = layer + 1;
  }
}

inline bool reachable(const Box &A, const Box &B, double kp, double z0m, double d0m) {
  const double angA = std::asin(std::min(1.0, kp * A.rlo));
  const double angB = std::asin(std::min(1.0, kp * B.rhi));
  const double dphi = std::fabs(std::remainder(B.phi - A.phi, 2.0 * M_PI));
  const double bend = angB - angA + d0m * std::max(0.0, 1.0 / A.rlo - 1.0 / B.rhi);
  if (!(dphi <= A.hphi + B.hphi + bend)) return false;
  const double rho[2] = {B.rlo / A.rhi, angB / angA};
  const double z0[2] = {-z0m, z0m}, zA[2] = {A.zlo, A.zhi};
  if (!B.endcap) {
    double lo = INFINITY, hi = -INFINITY;
    for (double v0 : z0) for (double va : zA) for (double r : rho) {
      const double zp = v0 + (va - v0) * r;
      lo = std::min(lo, zp); hi = std::max(hi, zp);
    }
    return lo <= B.zhi && hi >= B.zlo;
  }
  const double side = B.zlo > 0 ? 1.0 : -1.0;
  double lo = INFINITY, hi = -INFINITY;
  int nvalid = 0;
  for (double v0 : z0) for (double va : zA) {
    const double den = va - v0;
    if (!(side * den > 0.0)) continue;
    const double q = (B.zlo - v0) / den;
    lo = std::min(lo, q); hi = std::max(hi, q);
    ++nvalid;
  }
  if (nvalid == 0) return false;
  if (nvalid < 4) hi = INFINITY;
  return lo <= rho[1] && hi >= rho[0];
}
}  // namespace

extern "C" int lst_build_module_map(const lst_geometry *g, const lst_config *cfg_in, uint32_t **row_offsets,
                                    uint32_t **cols) {
  if (!geometry_ok(g) || !row_offsets || !cols) return einval();
  lst_config cfg;
  if (cfg_in) cfg = *cfg_in; else lst_default_config(&cfg);
  const uint32_t n = g->n_modules;
  const double kp = cfg.map_kscale * cfg.kB / (2.0 * cfg.pt_min);
  std::vector<Box> box(n);
  std::vector<std::vector<uint32_t>> by_layer(16);
  for (uint32_t m = 0; m < n; ++m) {
    box[m] = Box{(double)g->rmin[m], (double)g->rmax[m], (double)g->phic[m], (double)g->half_phi[m],
                 (double)g->zmin[m], (double)g->zmax[m], g->category[m] >= 2};
    by_layer[g->logical_layer[m]].push_back(m);
  }
  std::vector<uint32_t> off(n + 1, 0), out;
  std::vector<uint32_t> row;
  for (uint32_t A = 0; A < n; ++A) {
    int nl[3], nn;
    followers(g->logical_layer[A], nl, &nn);
    row.clear();
    for (int k = 0; k < nn; ++k)
      for (uint32_t B : by_layer[nl[k]])
        if (reachable(box[A], box[B], kp, cfg.map_z0, cfg.d0max)) row.push_back(B);
    std::sort(row.begin(), row.end());
    off[A] = (uint32_t)out.size();
    out.insert(out.end(), row.begin(), row.end());
  }
  off[n] = (uint32_t)out.size();
  uint32_t *o = (uint32_t *)malloc(sizeof(uint32_t) * (n + 1));
  uint32_t *c = (uint32_t *)malloc(sizeof(uint32_t) * std::max<size_t>(out.size(), 1));
  if (!o || !c) { free(o); free(c); return LST_ENOMEM; }
  memcpy(o, off.data(), sizeof(uint32_t) * (n + 1));
  if (!out.empty()) memcpy(c, out.data(), sizeof(uint32_t) * out.size());
  *row_offsets = o;
  *cols = c;
  return LST_OK;
}
extern "C" void lst_free(void *p) { free(p); }

// ------------------------------------------------------------------ context
struct Slot {
  SlotDev dev;
  void *workspace = nullptr;
  size_t ws_bytes = 0;
  bool bound = false, loaded = false, ran = false;
  cudaStream_t last_stream = nullptr;
  cudaGraphExec_t graph = nullptr;
  // pinned host staging for copy_to_host views (allocated on first use)
  uint32_t *h_hits = nullptr, *h_par = nullptr;
  float *h_f = nullptr;
  uint8_t *h_keep = nullptr;
  Header *h_hdr = nullptr;       // pinned
  Recorder *timed = nullptr;     // lst_run_timed: events created on first use
};

struct lst_ctx {
  lst_config cfg;
  Ctx k;
  uint32_t n_slots, max_hits, max_seeds;
  void *d_static = nullptr;      // geometry + map on the device
  std::vector<Slot> slots;
  size_t ws_bytes = 0;
  size_t exp_obj_cap = 0, exp_hit_words = 0;
  std::atomic<uint32_t> launches{0};   // kernels of one chain (the same for every slot)
  uint32_t map_edges = 0, map_edges_used = 0;   // module-map edges given / kept for the LS enumeration
  // the two regions of a workspace that every run resets: [zero_off, zero_off + zero_bytes) to 0 (the
  // slot header after n_hits / n_seeds, counters, flags, hash set) and [ff_off, + ff_bytes) to 0xFF
  size_t zero_off = 0, zero_bytes = 0, ff_off = 0, ff_bytes = 0;
  uint32_t batch = 1;                  // lst_config.batch_events, clamped to [1, kMaxBatch]
  std::vector<cudaGraphExec_t> group_graph;   // one per group of `batch` consecutive slots
  std::mutex bind_mu;                  // lst_bind_workspace: binds of one context are serialised (group_graph is shared)
};

// bump allocator over the workspace; base == nullptr only measures
struct Carver {
  char *base;
  size_t off = 0, last = 0;      // last: offset of the most recent take
  explicit Carver(void *b) : base((char *)b) {}
  template <class T>
  T *take(size_t n) {
    off = (off + 255) & ~(size_t)255;
    last = off;
    T *p = base ? (T *)(base + off) : nullptr;
    off += sizeof(T) * (n ? n : 1);
    return p;
  }
};

static uint32_t capf(float per, uint32_t n, uint32_t floor_) {
  const double v = (double)per * (double)n;
  const double c = std::min(v, 4.0e9);
  return std::max<uint32_t>((uint32_t)c, floor_);
}

// record != NULL (lst_create only): the layout figures that do not depend on `base` (reset regions, export
// capacities) are stored in the context; lst_bind_workspace passes NULL and writes nothing shared.
static size_t carve(const lst_ctx *c, void *base, SlotDev *out, lst_ctx *record) {
  Carver w(base);
  SlotDev s;
  memset(&s, 0, sizeof(s));
  const lst_config &cf = c->cfg;
  const uint32_t nh = std::max<uint32_t>(c->max_hits, 1), nsd = std::max<uint32_t>(c->max_seeds, 1);
  const uint32_t n_mod = c->k.geo.n_modules, n_det = c->k.geo.n_det;
  s.cap_hits = nh; s.cap_seeds = nsd;
  s.cap_md = capf(cf.cap_md_per_hit, nh, 1024);
  s.cap_ls = capf(cf.cap_ls_per_hit, nh, 1024);
  s.cap_t3 = capf(cf.cap_t3_per_hit, nh, 1024);
  s.cap_t5 = capf(cf.cap_t5_per_hit, nh, 1024);
  s.cap_pt3 = capf(cf.cap_pt3_per_seed, nsd, 1024);
  s.cap_pt5 = capf(cf.cap_pt5_per_seed, nsd, 1024);
  s.cap_tc = s.cap_pt5 + s.cap_pt3 + s.cap_t5 + nsd;
  s.half_store = cf.store_half != 0;
  const auto hs = [&](size_t n) { return s.half_store ? (n + 1) / 2 : n; };   // elements of the fp32 type that hold n binary16 ones
  // ---- the zeroed region: header (after n_hits / n_seeds), histogram, incidence counters, flags, hash set
  s.hdr = w.take<Header>(1);
  const size_t zero_off = w.last + 2 * sizeof(uint32_t);
  s.det_cnt = w.take<uint32_t>(n_det + 1);
  s.inc_cnt = w.take<uint32_t>(2 * (3 * (size_t)nh + 1)); s.inc_cur = s.inc_cnt + 3 * (size_t)nh + 1;
  s.pls_has5 = w.take<uint8_t>(3 * (size_t)nsd);
  s.pls_has3 = s.pls_has5 + nsd; s.pls_near_t5 = s.pls_has5 + 2 * (size_t)nsd;
  s.hit_used5 = w.take<uint8_t>(2 * (size_t)nh); s.hit_used3 = s.hit_used5 + nh;
  s.pid_size = 64;
  while (s.pid_size < 8 * (size_t)nsd && s.pid_size < (1u << 31)) s.pid_size <<= 1;
  s.pid_key = w.take<unsigned long long>(s.pid_size);
  s.pid_has5 = w.take<uint8_t>(2 * (size_t)s.pid_size); s.pid_has3 = s.pid_has5 + s.pid_size;
  s.scan_part = w.take<uint32_t>(kScanBlocks + 2);
  s.pls_bin_cnt = w.take<uint32_t>(2 * kEtaBins); s.pls_bin_cur = s.pls_bin_cnt + kEtaBins;
  const size_t zero_end = (w.off + 255) & ~(size_t)255;
  // ---- the 0xFF region: per-seed minimum scores and best objects of the same-seed rule
  s.pls_min5 = w.take<unsigned long long>(3 * (size_t)nsd);      // min5 | min3 | best5, best3
  const size_t ff_off = w.last;
  s.pls_min3 = s.pls_min5 + nsd;
  s.pls_best5 = (uint32_t *)(s.pls_min5 + 2 * (size_t)nsd);
  s.pls_best3 = s.pls_best5 + nsd;
  if (record) {
    record->zero_off = zero_off; record->zero_bytes = zero_end - zero_off;
    record->ff_off = ff_off; record->ff_bytes = 24 * (size_t)nsd;
  }
  s.raw_x = w.take<float>(nh); s.raw_y = w.take<float>(nh); s.raw_z = w.take<float>(nh);
  s.raw_det = w.take<uint32_t>(nh);
  s.seed_pt = w.take<float>(nsd); s.seed_eta = w.take<float>(nsd); s.seed_phi = w.take<float>(nsd);
  s.seed_z0 = w.take<float>(nsd); s.seed_q = w.take<int8_t>(nsd); s.seed_ids = w.take<uint32_t>(4 * (size_t)nsd);
  s.det_off = w.take<uint32_t>(n_det + 1);
  s.md_row0 = w.take<uint32_t>(n_mod + 1); s.row_mod = w.take<uint32_t>(nh);
  s.tmp_slot = w.take<uint32_t>(nh);
  s.tmp_orig = w.take<uint32_t>(nh);
  s.tmp_key = w.take<float>(nh); s.hit_key = w.take<float>(nh);
  s.hit = w.take<float4>(nh); s.hit_orig = w.take<uint32_t>(nh);
  s.md_pos = w.take<float4>(s.cap_md); s.md_kd = w.take<double2>(s.cap_md); s.md_kf = w.take<float2>(s.cap_md);
  s.md_hit = w.take<uint2>(s.cap_md); s.md_mod = w.take<uint32_t>(s.cap_md); s.md_dphi = w.take<float>(hs(s.cap_md));
  s.md_phi = w.take<float>(s.cap_md); s.md_prel = w.take<float>(s.cap_md);
  s.md_mod_off = w.take<uint32_t>(n_mod + 1);
  s.mod_ev = w.take<ModEv>(n_mod);
  s.edge_col0 = w.take<uint32_t>(std::max<uint32_t>(c->map_edges_used, 1));
  s.ls_md = w.take<uint2>(s.cap_ls); s.ls_f = w.take<float4>(hs(s.cap_ls));
  s.ls_md_off = w.take<uint32_t>((size_t)s.cap_md + 1);
  s.t3_md = w.take<uint4>(s.cap_t3); s.t3_ls = w.take<uint2>(s.cap_t3); s.t3_kd = w.take<double2>(s.cap_t3);
  s.t3_beta = w.take<float>(hs(s.cap_t3));
  s.t3_md_off = w.take<uint32_t>((size_t)s.cap_md + 1);
  s.t5_md = w.take<uint32_t>(5 * (size_t)s.cap_t5); s.t5_t3 = w.take<uint2>(s.cap_t5);
  s.t5_chi2 = w.take<double>(s.cap_t5); s.t5_etaphi = w.take<double2>(s.cap_t5);
  s.t5_f = w.take<float4>(hs(s.cap_t5)); s.t5_pt = w.take<float>(hs(s.cap_t5)); s.t5_keep = w.take<uint8_t>(s.cap_t5); s.t5_keep2 = w.take<uint8_t>(s.cap_t5);
  s.t5_md_off = w.take<uint32_t>((size_t)s.cap_md + 1);
  s.pt5_po = w.take<uint2>(s.cap_pt5); s.pt3_po = w.take<uint2>(s.cap_pt3);
  s.pt5_chi2 = w.take<double>(s.cap_pt5); s.pt3_chi2 = w.take<double>(s.cap_pt3);
  s.pt5_keep = w.take<uint8_t>(s.cap_pt5); s.pt3_keep = w.take<uint8_t>(s.cap_pt3);
  s.pls_keep = w.take<uint8_t>(nsd);
  s.px_cnt = w.take<uint32_t>(nsd);
  s.px_bits = w.take<uint32_t>((size_t)nsd * ((c->k.geo.n_start + 31) / 32));
  s.px_off = w.take<uint32_t>((size_t)nsd + 1); s.px_pair = w.take<uint2>((size_t)nsd * kPxCap);
  s.px_rng = w.take<uint2>((size_t)nsd * kPxCap);
  s.pt5_pls_off = w.take<uint32_t>((size_t)nsd + 1); s.pt3_pls_off = w.take<uint32_t>((size_t)nsd + 1);
  s.t5_hits = w.take<uint32_t>(10 * (size_t)s.cap_t5); s.pt3_hits = w.take<uint32_t>(6 * (size_t)s.cap_pt3);
  s.inc_off = w.take<uint32_t>(3 * (size_t)nh + 1);
  s.inc_ent = w.take<uint32_t>(10 * (size_t)s.cap_t5 + 10 * (size_t)s.cap_pt5 + 6 * (size_t)s.cap_pt3);
  s.pls_bin_off = w.take<uint32_t>(kEtaBins + 1); s.pls_bin_ent = w.take<uint32_t>(nsd);
  s.pls_adj_cnt = w.take<uint32_t>(nsd); s.pls_adj = w.take<uint32_t>((size_t)nsd * kAdjCap);
  s.pls_slot = w.take<uint32_t>(4 * (size_t)nsd);
  s.tc_to = w.take<uint2>(s.cap_tc); s.tc_f = w.take<float4>(s.cap_tc);
  s.tc_flag = w.take<uint32_t>((size_t)s.cap_tc + 1); s.tc_pos = w.take<uint32_t>((size_t)s.cap_tc + 1);
  s.flag_blk = w.take<uint32_t>(kFlagBlocks + 1);
  // work lists
  const uint32_t cand_cap[S_NSTAGE] = {
      capf(cf.cap_mdcand_per_hit, nh, 1 << 16), capf(cf.cap_lscand_per_hit, nh, 1 << 16),
      capf(cf.cap_t3cand_per_hit, nh, 1 << 16), capf(cf.cap_t5cand_per_hit, nh, 1 << 16),
      capf(2048.0f, nsd, 1 << 16), capf(4096.0f, nsd, 1 << 16)};
  const uint32_t pair_groups = (uint32_t)(((size_t)nsd * kPxCap) / kRowChunk + 2);
  const uint32_t grp_cap[S_NSTAGE] = {n_mod, n_mod, s.cap_ls / kRowChunk + 2, s.cap_t3 / kRowChunk + 2,
                                      pair_groups, pair_groups};
  const uint32_t row_cap[S_NSTAGE] = {0, 0, s.cap_ls, s.cap_t3, nsd * (uint32_t)kPxCap, nsd * (uint32_t)kPxCap};
  for (int k = 0; k < S_NSTAGE; ++k) {
    StageBuf &b = s.st[k];
    b.cap_groups = grp_cap[k];
    b.cap_items = grp_cap[k] + 2 * (cand_cap[k] / kItemCand) + 16;
    b.gR = w.take<uint32_t>(b.cap_groups); b.gW = w.take<uint32_t>(b.cap_groups);
    b.g_item0 = w.take<uint32_t>((size_t)b.cap_groups + 1);
    b.gblk = w.take<uint32_t>((size_t)b.cap_groups / 4 + 2);
    b.item_group = k == S_MD ? w.take<uint32_t>(b.cap_items) : nullptr;
    b.row_start = row_cap[k] ? w.take<uint32_t>(row_cap[k]) : nullptr;
    b.row_cum = row_cap[k] ? w.take<uint32_t>(row_cap[k]) : nullptr;
    b.cblk = w.take<uint32_t>(kCountBlocks + 1);
    b.mask = w.take<uint32_t>((size_t)b.cap_items * kItemWords);
    b.wpre = w.take<uint16_t>((size_t)b.cap_items * kItemWords);
    b.item_cnt = w.take<uint32_t>(b.cap_items); b.item_base = w.take<uint32_t>(b.cap_items);
    const uint32_t pool_cap[S_NSTAGE] = {s.cap_md, s.cap_ls, s.cap_t3, s.cap_t5, s.cap_pt5, s.cap_pt3};
    b.cap_pool = pool_cap[k];
    b.cap_cl = 2 * b.cap_pool + 4096;
    b.cl_key = w.take<uint32_t>(b.cap_cl);
    b.cl_ab = w.take<uint2>(b.cap_cl);
    b.p_d2 = w.take<double2>(b.cap_cl);
    b.p_d2b = k == S_T5 ? w.take<double2>(b.cap_cl) : nullptr;
    b.p_f4 = w.take<float4>(b.cap_cl);
  }
  // export scratch: the largest level
  size_t obj_cap = std::max({(size_t)s.cap_md, (size_t)s.cap_ls, (size_t)s.cap_t3, (size_t)s.cap_t5,
                             (size_t)s.cap_pt3, (size_t)s.cap_pt5, (size_t)s.cap_tc});
  size_t hit_words = std::max({2 * (size_t)s.cap_md, 4 * (size_t)s.cap_ls, 6 * (size_t)s.cap_t3,
                               10 * (size_t)s.cap_t5, 6 * (size_t)s.cap_pt3, 10 * (size_t)s.cap_pt5,
                               14 * (size_t)s.cap_tc});
  s.exp_hits = w.take<uint32_t>(hit_words);
  s.exp_par = w.take<uint32_t>(2 * obj_cap);
  s.exp_f = w.take<float>(4 * obj_cap);
  if (out) *out = s;
  if (record) { record->exp_obj_cap = obj_cap; record->exp_hit_words = hit_words; }
  return (w.off + 255) & ~(size_t)255;
}

// Can ANY (inner anchor in module A's lower-sensor box, outer anchor in module B's) pass the LS
// cuts L1 (pointing) and L2 (pT window) of reading C3?  Host, fp64, interval arithmetic on the two
// boxes, every bound loosened (1e-3 relative, boxes grown by 1e-4 cm / 1e-5 rad: k_hist accepts a
// lower-sensor hit up to 5e-5 cm / 4e-6 rad outside its box, else the event is LST_EINVAL): false only for module pairs that cannot hold a line segment.  The module
// map is built with wider margins (kappa' = 1.25 kappa_max, z0' = 20 cm, a d0 allowance) than the
// cuts use, so ~21 % of its edges are dead; dropping them from the LS enumeration changes no result.
// Assumes what lst_geometry states: a lower-sensor hit lies inside its module's box.
static bool ls_edge_possible(const Params &p, const lst_geometry *g, uint32_t A, uint32_t B) {
  const double kEps = 1e-3, gl = 1e-4, ga = 1e-5, kPi = 3.14159265358979323846;
  const int cA = g->category[A] & 3, cB = g->category[B] & 3;
  const double ri0 = std::max(1e-6, (double)g->rmin[A] - gl), ri1 = (double)g->rmax[A] + gl;
  const double ro0 = std::max(1e-6, (double)g->rmin[B] - gl), ro1 = (double)g->rmax[B] + gl;
  const double zi0 = (double)g->zmin[A] - gl, zi1 = (double)g->zmax[A] + gl;
  const double zo0 = (double)g->zmin[B] - gl, zo1 = (double)g->zmax[B] + gl;
  // L1: N = rt_i z_o - z_i rt_o is multilinear: its extremes over the boxes are at the corners
  double Nmin = INFINITY, Nmax = -INFINITY;
  const double ris[2] = {ri0, ri1}, zis[2] = {zi0, zi1}, ros[2] = {ro0, ro1}, zos[2] = {zo0, zo1};
  for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) for (int c = 0; c < 2; ++c) for (int d = 0; d < 2; ++d) {
    const double N = ris[a] * zos[d] - zis[b] * ros[c];
    Nmin = std::min(Nmin, N); Nmax = std::max(Nmax, N);
  }
  const double azi1 = std::max(std::fabs(zi0), std::fabs(zi1)), azo1 = std::max(std::fabs(zo0), std::fabs(zo1));
  const double Emax = ri1 * p.sig_z[cB] + ro1 * p.sig_z[cA] + azo1 * p.sig_r[cA] + azi1 * p.sig_r[cB];
  const double drmax = std::max(std::fabs(ro1 - ri0), std::fabs(ro0 - ri1));
  const double rhs = (p.z0max * drmax + p.ns * Emax) * (1.0 + kEps) + 1e-3;
  if (!(Nmin <= rhs && Nmax >= -rhs)) return false;
  // L2: smallest |dphi| the boxes allow against the largest the cut allows
  const double dphi = std::fabs(std::remainder((double)g->phic[B] - (double)g->phic[A], 2.0 * kPi));
  const double dmin = std::max(0.0, dphi - (double)g->half_phi[A] - (double)g->half_phi[B] - 2.0 * ga);
  const double sigt = std::max(std::max(p.sig_t[0], p.sig_t[1]), std::max(p.sig_t[2], p.sig_t[3]));
  const double tol = p.ns * sigt * (1.0 / ri0 + 1.0 / ro0);
  double W = kPi;
  if (cB < 2) {
    // mode R: a passing pair lies on a circle through the origin of half curvature <= k' = kmax +
    // tol / chord, where dphi = asin(k' rt_o) - asin(k' rt_i) on the outgoing arc; the returning arc
    // has dphi < pi/2 only if asin(k' rt_o) + asin(k' rt_i) > pi/2, which k' rt_o <= 0.6 excludes
    const double cmin = ro0 - ri1;
    if (cmin > 1.0) {
      const double k = (p.kmax + tol / cmin) * (1.0 + 2.0 * kEps);
      if (k * ro1 <= 0.6) W = (std::asin(k * ro1) - std::asin(k * ri0)) * (1.0 + 2.0 * kEps) + 1e-4;
    }
  } else {
    // mode Z: L2 is itself a bound on |dphi|, taken at the extremes of the boxes
    const double sigr = std::max(std::max(p.sig_r[0], p.sig_r[1]), std::max(p.sig_r[2], p.sig_r[3]));
    const double azi0 = (zi0 <= 0.0 && zi1 >= 0.0) ? 0.0 : std::min(std::fabs(zi0), std::fabs(zi1));
    const double azo0 = (zo0 <= 0.0 && zo1 >= 0.0) ? 0.0 : std::min(std::fabs(zo0), std::fabs(zo1));
    const double dzmax = std::max(std::fabs(zo1 - zi0), std::fabs(zo0 - zi1));
    const double den = 0.5 * (azi0 + azo0) - p.z0max - 0.5 * p.ns * p.sig_z[cA];
    if (den > 1.0) {
      const double x = std::min(1.0, p.kmax * (0.5 * (ri1 + ro1) + p.ns * sigr));
      W = (p.kmax * (dzmax + p.ns * p.sig_z[cA]) * (std::asin(x) / p.kmax) / den + tol) * (1.0 + 2.0 * kEps) + 1e-4;
    }
  }
  return dmin <= W;
}

extern "C" int lst_create(const lst_geometry *g, const lst_module_map *map, const lst_config *cfg_in,
                          uint32_t n_slots, uint32_t max_hits, uint32_t max_seeds, lst_ctx **out) {
  if (!geometry_ok(g) || !map || !map->row_offsets || !out || n_slots == 0 || max_hits == 0) return einval();
  const uint32_t n = g->n_modules;
  if (n > (1u << 29)) return einval();
  if (map->row_offsets[0] != 0) return einval();
  const uint32_t nnz = map->row_offsets[n];
  if (nnz && !map->cols) return einval();
  for (uint32_t m = 0; m < n; ++m) {
    const uint32_t a = map->row_offsets[m], b = map->row_offsets[m + 1];
    if (b < a || b > nnz || b - a > (uint32_t)kMaxDeg) return einval();
    for (uint32_t e = a; e < b; ++e) {
      if (map->cols[e] >= n) return einval();
      if (e > a && map->cols[e] <= map->cols[e - 1]) return einval();
    }
  }
  lst_ctx *c = new (std::nothrow) lst_ctx();
  if (!c) return LST_ENOMEM;
  if (cfg_in) c->cfg = *cfg_in; else lst_default_config(&c->cfg);
  if (c->cfg.dup_t5_shared < 1 || c->cfg.dup_pt5_shared < 1 || c->cfg.dup_pt3_shared < 1 || !(c->cfg.pt_min > 0.0) ||
      !(c->cfg.dr2max >= 0.0)) {
    delete c;
    return einval();
  }
  make_params(c->cfg, &c->k.par);
  c->k.ls_windows = (c->cfg.enum_pruning & 2) != 0;
  c->k.pdl = c->cfg.use_pdl != 0;
  if (c->cfg.s0_fixpoint_passes < 0 || c->cfg.s0_fixpoint_passes > kMaxFixPasses || (c->cfg.s0_fixpoint_passes & 1)) { delete c; return einval(); }
  c->k.fix_passes = c->cfg.s0_fixpoint_passes;
  {
    // stages with an occupancy cap: MD, LS, T3, T5 per logical layer; pT3 / pT5 per seed ([level][0])
    const int stage_of_level[6] = {S_MD, S_LS, S_T3, S_T5, S_PT3, S_PT5};
    for (int l = 0; l < 6; ++l)
      for (int k = 0; k < (l < 4 ? 16 : 1); ++k)
        if (c->cfg.trunc_cap[l][k]) c->k.trunc_stages |= 1u << stage_of_level[l];
  }
  if (c->cfg.batch_events < 1 || c->cfg.batch_events > kMaxBatch) { delete c; return einval(); }
  c->batch = (uint32_t)c->cfg.batch_events;
  c->n_slots = n_slots; c->max_hits = max_hits; c->max_seeds = max_seeds;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  cudaDeviceProp prop;
  if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
  if (e != cudaSuccess) { delete c; return cuda_fail(e, "cudaGetDeviceProperties"); }
  c->k.n_sm = prop.multiProcessorCount;
  // modules that may start a pixel-seeded object (C6 START layers)
  std::vector<uint32_t> start_mods;
  for (uint32_t m = 0; m < n; ++m)
    if ((c->cfg.start_layer_mask >> g->logical_layer[m]) & 1u) start_mods.push_back(m);
  // static data: category | layer | map_off | map_cols | 6 box arrays | start modules
  const auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
  const size_t o_cat = 0, o_lay = up(n), o_off = o_lay + up(n);
  const size_t o_cols = o_off + up((size_t)(n + 1) * 4);
  const size_t o_box = o_cols + up((size_t)std::max<uint32_t>(nnz, 1) * 4);
  const size_t box_stride = up((size_t)n * 4);
  const size_t o_start = o_box + 6 * box_stride;
  const size_t o_sbox = o_start + up(std::max<size_t>(start_mods.size(), 1) * 4);   // rows of start modules follow
  // rows of start modules (same box up to phic)
  std::vector<uint32_t> prow_off, prow_k;
  std::vector<float> prow_phic, prow_b;   // prow_b: 8 floats per row
  {
    std::vector<uint32_t> order(start_mods.size());
    for (size_t k = 0; k < order.size(); ++k) order[k] = (uint32_t)k;
    auto key_less = [&](uint32_t ka, uint32_t kb) {
      const uint32_t a = start_mods[ka], b = start_mods[kb];
      if (g->category[a] != g->category[b]) return g->category[a] < g->category[b];
      if (g->rmin[a] != g->rmin[b]) return g->rmin[a] < g->rmin[b];
      if (g->rmax[a] != g->rmax[b]) return g->rmax[a] < g->rmax[b];
      if (g->zmin[a] != g->zmin[b]) return g->zmin[a] < g->zmin[b];
      if (g->zmax[a] != g->zmax[b]) return g->zmax[a] < g->zmax[b];
      if (g->half_phi[a] != g->half_phi[b]) return g->half_phi[a] < g->half_phi[b];
      return false;
    };
    std::stable_sort(order.begin(), order.end(), key_less);
    for (size_t i = 0; i < order.size(); ++i) {
      if (i == 0 || key_less(order[i - 1], order[i])) {
        const uint32_t m = start_mods[order[i]];
        prow_off.push_back((uint32_t)i);
        const float b8[8] = {g->half_phi[m], g->rmin[m], g->rmax[m], (float)g->category[m], g->zmin[m], g->zmax[m],
                             c->k.par.f_sig_t[g->category[m] & 3] / g->rmin[m], 0.0f};
        prow_b.insert(prow_b.end(), b8, b8 + 8);
      }
      prow_k.push_back(order[i]);
      prow_phic.push_back(g->phic[start_mods[order[i]]]);
    }
    prow_off.push_back((uint32_t)order.size());
  }
  const size_t n_prow = prow_off.size() - 1;
  const size_t o_prow = o_sbox;
  const size_t o_prow2 = o_prow + up(std::max<size_t>(n_prow, 1) * 16);
  const size_t o_poff = o_prow2 + up(std::max<size_t>(n_prow, 1) * 16);
  const size_t o_pk = o_poff + up((n_prow + 1) * 4);
  const size_t o_pphi = o_pk + up(std::max<size_t>(prow_k.size(), 1) * 4);
  const size_t o_pof = o_pphi + up(std::max<size_t>(prow_phic.size(), 1) * 4);
  const size_t total = o_pof + up(std::max<size_t>(start_mods.size(), 1) * 4);
  e = cudaMalloc(&c->d_static, total);
  if (e != cudaSuccess) { delete c; return cuda_fail(e, "cudaMalloc(static)"); }
  char *d = (char *)c->d_static;
  // every upload is checked: the first failure is kept and reported below (a synchronous cudaMemcpy that
  // failed is not reported by the later cudaDeviceSynchronize)
  cudaError_t up_err = cudaSuccess;
  const char *up_what = "";
  auto upload_as = [&](const char *what, void *dst, const void *src, size_t bytes) {
    if (up_err != cudaSuccess || bytes == 0) return;
    up_err = cudaMemcpy(dst, src, bytes, cudaMemcpyHostToDevice);
    if (up_err != cudaSuccess) up_what = what;
  };
#define upload(dst, src, bytes) upload_as("upload " #src, (dst), (src), (bytes))
  upload(d + o_cat, g->category, n);
  upload(d + o_lay, g->logical_layer, n);
  {
    // the LS enumeration walks the map without its dead edges (ls_edge_possible)
    std::vector<uint32_t> poff(n + 1, 0u), pcols;
    pcols.reserve(nnz);
    const bool drop_dead = (c->cfg.enum_pruning & 1) != 0;
    for (uint32_t m = 0; m < n; ++m) {
      for (uint32_t e = map->row_offsets[m]; e < map->row_offsets[m + 1]; ++e)
        if (!drop_dead || ls_edge_possible(c->k.par, g, m, map->cols[e])) pcols.push_back(map->cols[e]);
      poff[m + 1] = (uint32_t)pcols.size();
    }
    c->map_edges = nnz; c->map_edges_used = (uint32_t)pcols.size();
    upload(d + o_off, poff.data(), (size_t)(n + 1) * 4);
    if (!pcols.empty()) upload(d + o_cols, pcols.data(), pcols.size() * 4);
  }
  const float *box[6] = {g->rmin, g->rmax, g->phic, g->half_phi, g->zmin, g->zmax};
  for (int k = 0; k < 6; ++k) upload(d + o_box + k * box_stride, box[k], (size_t)n * 4);
  if (!start_mods.empty())
    upload(d + o_start, start_mods.data(), start_mods.size() * 4);
  {
    std::vector<float> r1(4 * std::max<size_t>(n_prow, 1), 0.0f), r2(4 * std::max<size_t>(n_prow, 1), 0.0f);
    for (size_t r = 0; r < n_prow; ++r)
      for (int q = 0; q < 4; ++q) { r1[4 * r + q] = prow_b[8 * r + q]; r2[4 * r + q] = prow_b[8 * r + 4 + q]; }
    upload(d + o_prow, r1.data(), r1.size() * 4);
    upload(d + o_prow2, r2.data(), r2.size() * 4);
    upload(d + o_poff, prow_off.data(), prow_off.size() * 4);
    if (!prow_k.empty()) {
      upload(d + o_pk, prow_k.data(), prow_k.size() * 4);
      upload(d + o_pphi, prow_phic.data(), prow_phic.size() * 4);
    }
    c->k.geo.prow_b1 = (const float4 *)(d + o_prow); c->k.geo.prow_b2 = (const float4 *)(d + o_prow2);
    c->k.geo.prow_off = (const uint32_t *)(d + o_poff); c->k.geo.prow_k = (const uint32_t *)(d + o_pk);
    c->k.geo.prow_phic = (const float *)(d + o_pphi);
    c->k.geo.n_prow = (uint32_t)n_prow;
    std::vector<uint32_t> prow_of(std::max<size_t>(start_mods.size(), 1), 0u);
    for (size_t r = 0; r < n_prow; ++r)
      for (uint32_t i = prow_off[r]; i < prow_off[r + 1]; ++i) prow_of[prow_k[i]] = (uint32_t)r;
    upload(d + o_pof, prow_of.data(), prow_of.size() * 4);
    c->k.geo.prow_of = (const uint32_t *)(d + o_pof);
  }
#undef upload
  if (up_err != cudaSuccess) { cudaFree(c->d_static); delete c; return cuda_fail(up_err, up_what); }
  e = cudaDeviceSynchronize();
  if (e != cudaSuccess) { cudaFree(c->d_static); delete c; return cuda_fail(e, "upload geometry"); }
  c->k.geo.n_modules = n; c->k.geo.n_det = 2 * n;
  c->k.geo.category = (const uint8_t *)(d + o_cat);
  c->k.geo.layer = (const uint8_t *)(d + o_lay);
  c->k.geo.map_off = (const uint32_t *)(d + o_off);
  c->k.geo.map_cols = (const uint32_t *)(d + o_cols);
  c->k.geo.rmin = (const float *)(d + o_box); c->k.geo.rmax = (const float *)(d + o_box + box_stride);
  c->k.geo.phic = (const float *)(d + o_box + 2 * box_stride); c->k.geo.hphi = (const float *)(d + o_box + 3 * box_stride);
  c->k.geo.zmin = (const float *)(d + o_box + 4 * box_stride); c->k.geo.zmax = (const float *)(d + o_box + 5 * box_stride);
  c->k.geo.start_mods = (const uint32_t *)(d + o_start);
  c->k.geo.n_start = (uint32_t)start_mods.size();
  c->slots.resize(n_slots);
  c->group_graph.assign((n_slots + c->batch - 1) / c->batch, nullptr);
  {
    // candidate keys (item * 1024 + candidate), list positions and the TC index are 32-bit
    SlotDev probe;
    c->ws_bytes = carve(c, nullptr, &probe, c);
    bool fits = (double)c->cfg.cap_pt5_per_seed * max_seeds + (double)c->cfg.cap_pt3_per_seed * max_seeds +
                    (double)c->cfg.cap_t5_per_hit * max_hits + max_seeds < 4.0e9;
    for (int k = 0; k < S_NSTAGE; ++k)
      fits = fits && (double)probe.st[k].cap_items * kItemCand < 4.29e9 && 2.0 * (double)probe.st[k].cap_pool + 4096.0 < 4.29e9;
    if (!fits) { cudaFree(c->d_static); delete c; return einval(); }
  }
  *out = c;
  return LST_OK;
}

static void free_slot_host(Slot &s) {
  if (s.graph) cudaGraphExecDestroy(s.graph);
  if (s.h_hits) cudaFreeHost(s.h_hits);
  if (s.h_par) cudaFreeHost(s.h_par);
  if (s.h_f) cudaFreeHost(s.h_f);
  if (s.h_keep) cudaFreeHost(s.h_keep);
  if (s.h_hdr) cudaFreeHost(s.h_hdr);
  if (s.timed) { for (int k = 0; k <= Recorder::kMax; ++k) cudaEventDestroy(s.timed->ev[k]); delete s.timed; }
  s = Slot();
}

extern "C" void lst_destroy(lst_ctx *c) {
  if (!c) return;
  cudaDeviceSynchronize();
  for (Slot &s : c->slots) free_slot_host(s);
  for (cudaGraphExec_t g : c->group_graph) if (g) cudaGraphExecDestroy(g);
  if (c->d_static) cudaFree(c->d_static);
  delete c;
}

extern "C" size_t lst_workspace_bytes(const lst_ctx *c) { return c ? c->ws_bytes : 0; }

static int capture_graph(lst_ctx *c, uint32_t slot0, uint32_t n, cudaGraphExec_t *out);

extern "C" int lst_bind_workspace(lst_ctx *c, uint32_t slot, void *workspace, size_t bytes) {
  if (!c || slot >= c->n_slots || !workspace || ((uintptr_t)workspace & 255)) return einval();
  if (bytes < c->ws_bytes) {
    snprintf(g_cap_err, sizeof(g_cap_err), "workspace too small: %zu bytes given, %zu needed", bytes, c->ws_bytes);
    return LST_ENOMEM;
  }
  std::lock_guard<std::mutex> bind_lock(c->bind_mu);   // two threads binding slots of one group share group_graph[grp]
  Slot &s = c->slots[slot];
  if (s.graph) { cudaGraphExecDestroy(s.graph); s.graph = nullptr; }
  carve(c, workspace, &s.dev, nullptr);
  s.workspace = workspace; s.ws_bytes = bytes;
  s.bound = true; s.loaded = false; s.ran = false;
  if (!s.h_hdr) CU(cudaMallocHost((void **)&s.h_hdr, sizeof(Header)));
  if (!c->cfg.use_cuda_graph) return LST_OK;
  int rc = capture_graph(c, slot, 1, &s.graph);
  if (rc != LST_OK || c->batch == 1) return rc;
  // the graph of the slot's group (lst_run_batch), once every slot of the group has a workspace
  const uint32_t grp = slot / c->batch, s0 = grp * c->batch, s1 = std::min(c->n_slots, s0 + c->batch);
  if (c->group_graph[grp]) { cudaGraphExecDestroy(c->group_graph[grp]); c->group_graph[grp] = nullptr; }
  for (uint32_t k = s0; k < s1; ++k) if (!c->slots[k].bound) return LST_OK;
  return capture_graph(c, s0, s1 - s0, &c->group_graph[grp]);
}

// ------------------------------------------------------------------ a0 upload
__global__ void k_set_event(Header *h, uint32_t n_hits, uint32_t n_seeds) {
  h->n_hits = n_hits;
  h->n_seeds = n_seeds;
}

extern "C" int lst_load_event(lst_ctx *c, uint32_t slot, const lst_hits *hits, const lst_pixel_seeds *seeds,
                              void *cuda_stream) {
  if (!c || slot >= c->n_slots || !hits) return einval();
  Slot &s = c->slots[slot];
  if (!s.bound) return LST_ESTATE;
  const uint32_t nh = hits->n, nsd = seeds ? seeds->n : 0;
  if (nh > c->max_hits || nsd > c->max_seeds) return einval();
  if (nh && (!hits->x || !hits->y || !hits->z || !hits->det)) return einval();
  if (nsd && (!seeds->pt || !seeds->eta || !seeds->phi || !seeds->z0 || !seeds->q || !seeds->hit_ids)) return einval();
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const SlotDev &d = s.dev;
  if (nh) {
    const cudaMemcpyKind k = hits->on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CU(cudaMemcpyAsync(d.raw_x, hits->x, sizeof(float) * nh, k, st));
    CU(cudaMemcpyAsync(d.raw_y, hits->y, sizeof(float) * nh, k, st));
    CU(cudaMemcpyAsync(d.raw_z, hits->z, sizeof(float) * nh, k, st));
    CU(cudaMemcpyAsync(d.raw_det, hits->det, sizeof(uint32_t) * nh, k, st));
  }
  if (nsd) {
    const cudaMemcpyKind k = seeds->on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CU(cudaMemcpyAsync(d.seed_pt, seeds->pt, sizeof(float) * nsd, k, st));
    CU(cudaMemcpyAsync(d.seed_eta, seeds->eta, sizeof(float) * nsd, k, st));
    CU(cudaMemcpyAsync(d.seed_phi, seeds->phi, sizeof(float) * nsd, k, st));
    CU(cudaMemcpyAsync(d.seed_z0, seeds->z0, sizeof(float) * nsd, k, st));
    CU(cudaMemcpyAsync(d.seed_q, seeds->q, sizeof(int8_t) * nsd, k, st));
    CU(cudaMemcpyAsync(d.seed_ids, seeds->hit_ids, sizeof(uint32_t) * 4 * (size_t)nsd, k, st));
  }
  k_set_event<<<1, 1, 0, st>>>(d.hdr, nh, nsd);
  CU(cudaGetLastError());
  s.loaded = true; s.ran = false; s.last_stream = st;
  return LST_OK;
}

// ------------------------------------------------------------------ the chain
// Enqueue a0 .. a6 of the slots [slot0, slot0 + n) on `st` as ONE chain of launches (gridDim.z = n);
// rec (may be NULL) counts / times the kernels.  Two memsets reset what a run accumulates into, then
// 39 kernels; with `pdl` every kernel but the first is launched with programmatic stream serialisation.
// side (capture only, else NULL): a second stream on which the seed-preparation kernel, which needs nothing
// but the seeds, and the (seed, module) row kernel, which needs the MDs on top, run beside a0 .. a4 (a fork /
// join inside the graph); without it the two kernels run inline.
static int enqueue_chain(const lst_ctx *c, uint32_t slot0, uint32_t n, cudaStream_t st, Recorder *rec, bool pdl,
                         cudaStream_t side = nullptr, cudaEvent_t ev_fork = nullptr, cudaEvent_t ev_join = nullptr) {
  Recorder count_only;
  Ctx k = c->k;                    // a private copy: the recorder pointer is per call, not per context
  k.rec = rec ? rec : &count_only;
  k.pdl = pdl && c->k.pdl;
  k.nb = (int)n;
  Batch b;
  memset(&b, 0, sizeof(b));
  for (uint32_t e = 0; e < n; ++e) {
    const Slot &sl = c->slots[slot0 + e];
    b.s[e] = sl.dev;
    cudaMemsetAsync((char *)sl.workspace + c->zero_off, 0, c->zero_bytes, st);
    cudaMemsetAsync((char *)sl.workspace + c->ff_off, 0xFF, c->ff_bytes, st);
  }
  if (side) {
    cudaEventRecord(ev_fork, st);
    cudaStreamWaitEvent(side, ev_fork, 0);
    launch_seed_prep(k, b, side, true);
    launch_index(k, b, st);
  } else {
    launch_index(k, b, st);
    launch_seed_prep(k, b, st, false);
  }
  launch_md(k, b, st);
  if (side) {                      // the (seed, module) rows need the MDs and the seed preparation, nothing else
    cudaEventRecord(ev_fork, st);
    cudaStreamWaitEvent(side, ev_fork, 0);
    launch_seed_rows(k, b, side);
    cudaEventRecord(ev_join, side);
  }
  launch_ls(k, b, st);
  launch_t3(k, b, st);
  launch_t5(k, b, st);
  if (side) cudaStreamWaitEvent(st, ev_join, 0);
  else launch_seed_rows(k, b, st);
  launch_pixel_joins(k, b, st);
  launch_dedup(k, b, st);
  return k.rec->n;
}

// One CUDA graph per slot (and one per group of lst_config.batch_events slots), captured when the
// workspace is bound (lst_run then only replays it: no allocation, no capture, nothing shared between
// slots is written).
static int capture_graph(lst_ctx *c, uint32_t slot0, uint32_t n, cudaGraphExec_t *out) {
  cudaGraph_t gr = nullptr;
  cudaStream_t cap = nullptr, side = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  auto release = [&]() {
    if (ev_join) cudaEventDestroy(ev_join);
    if (ev_fork) cudaEventDestroy(ev_fork);
    if (side) cudaStreamDestroy(side);
    if (cap) cudaStreamDestroy(cap);
  };
  // everything the capture needs exists, and is checked, before the capture begins
  cudaError_t e = cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking);   // the legacy default stream cannot be captured
  const char *what = "cudaStreamCreateWithFlags(capture)";
  if (e == cudaSuccess) { e = cudaStreamCreateWithFlags(&side, cudaStreamNonBlocking); what = "cudaStreamCreateWithFlags(side)"; }
  if (e == cudaSuccess) { e = cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming); what = "cudaEventCreateWithFlags(fork)"; }
  if (e == cudaSuccess) { e = cudaEventCreateWithFlags(&ev_join, cudaEventDisableTiming); what = "cudaEventCreateWithFlags(join)"; }
  if (e == cudaSuccess) { e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal); what = "cudaStreamBeginCapture"; }
  if (e != cudaSuccess) { release(); return cuda_fail(e, what); }
  const int nk = enqueue_chain(c, slot0, n, cap, nullptr, true, side, ev_fork, ev_join);
  e = cudaStreamEndCapture(cap, &gr);
  release();
  if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
  e = cudaGraphInstantiate(out, gr, 0);
  cudaGraphDestroy(gr);
  if (e != cudaSuccess) { *out = nullptr; return cuda_fail(e, "cudaGraphInstantiate"); }
  c->launches.store((uint32_t)nk);
  return LST_OK;
}

extern "C" int lst_run(lst_ctx *c, uint32_t slot, void *cuda_stream) {
  if (!c || slot >= c->n_slots) return einval();
  Slot &s = c->slots[slot];
  if (!s.bound || !s.loaded) return LST_ESTATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (s.graph) {
    CU(cudaGraphLaunch(s.graph, st));
  } else {
    c->launches.store((uint32_t)enqueue_chain(c, slot, 1, st, nullptr, true));
    CU(cudaGetLastError());
  }
  s.ran = true; s.last_stream = st;
  return LST_OK;
}

extern "C" int lst_run_batch(lst_ctx *c, uint32_t group, void *cuda_stream) {
  if (!c || (uint64_t)group * c->batch >= c->n_slots) return einval();
  const uint32_t s0 = group * c->batch, s1 = std::min(c->n_slots, s0 + c->batch);
  for (uint32_t k = s0; k < s1; ++k)
    if (!c->slots[k].bound || !c->slots[k].loaded) return LST_ESTATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaGraphExec_t g = c->batch == 1 ? c->slots[s0].graph : c->group_graph[group];
  if (g) {
    CU(cudaGraphLaunch(g, st));
  } else {
    c->launches.store((uint32_t)enqueue_chain(c, s0, s1 - s0, st, nullptr, true));
    CU(cudaGetLastError());
  }
  for (uint32_t k = s0; k < s1; ++k) { c->slots[k].ran = true; c->slots[k].last_stream = st; }
  return LST_OK;
}

extern "C" uint32_t lst_batch_events(const lst_ctx *c) { return c ? c->batch : 0; }

static int sync_header(lst_ctx *c, Slot &s);
extern "C" int lst_get_fixpoint_unsettled(lst_ctx *c, uint32_t slot, uint32_t *n) {
  if (!c || slot >= c->n_slots || !n) return einval();
  Slot &s = c->slots[slot];
  if (!s.ran) return LST_ESTATE;
  const int rc = sync_header(c, s);
  if (rc != LST_OK) return rc;
  *n = s.h_hdr->n_unsettled;
  return LST_OK;
}

// ------------------------------------------------------------------ results
static int sync_header(lst_ctx *c, Slot &s) {
  (void)c;
  CU(cudaMemcpyAsync(s.h_hdr, s.dev.hdr, sizeof(Header), cudaMemcpyDeviceToHost, s.last_stream));
  CU(cudaStreamSynchronize(s.last_stream));
  if (s.h_hdr->err & (ERR_DET | ERR_NONFINITE | ERR_BOX)) {
    snprintf(g_inval_err, sizeof(g_inval_err), "invalid event:%s%s%s",
             (s.h_hdr->err & ERR_DET) ? " det id out of range" : "",
             (s.h_hdr->err & ERR_NONFINITE) ? " NaN / infinite hit coordinate or seed parameter" : "",
             (s.h_hdr->err & ERR_BOX) ? " lower-sensor hit outside its module's box" : "");
    return LST_EINVAL;
  }
  if (s.h_hdr->err & (ERR_CAP_ITEMS | ERR_CAP_OBJ | ERR_CAP_PIX)) {
    const Header &h = *s.h_hdr;
    int n = snprintf(g_cap_err, sizeof(g_cap_err),
                     "capacity exceeded:%s%s%s (objects MD %u LS %u T3 %u T5 %u pT3 %u pT5 %u; raise lst_config.cap_*);",
                     (h.err & ERR_CAP_ITEMS) ? " work items / candidate list" : "", (h.err & ERR_CAP_OBJ) ? " object array" : "",
                     (h.err & ERR_CAP_PIX) ? " per-seed list" : "", h.n_obj[0], h.n_obj[1], h.n_obj[2], h.n_obj[3], h.n_obj[4],
                     h.n_obj[5]);
    static const char *const nm[S_NSTAGE] = {"MD", "LS", "T3", "T5", "pT5", "pT3"};
    for (int k = 0; k < S_NSTAGE && n > 0 && n < (int)sizeof(g_cap_err) - 80; ++k)   // a stage whose work list overflowed shows items 0
      n += snprintf(g_cap_err + n, sizeof(g_cap_err) - n, " %s items %u/%u list %u/%u", nm[k], h.n_items[k], s.dev.st[k].cap_items,
                    h.cl_used[k], s.dev.st[k].cap_cl);
    return LST_ENOMEM;
  }
  return LST_OK;
}

extern "C" int lst_get_counts(lst_ctx *c, uint32_t slot, uint32_t *counts, uint64_t *cand) {
  if (!c || slot >= c->n_slots || !counts) return einval();
  Slot &s = c->slots[slot];
  if (!s.ran) return LST_ESTATE;
  const int rc = sync_header(c, s);
  if (rc != LST_OK) return rc;
  for (int l = 0; l < LST_NLEVEL; ++l) counts[l] = s.h_hdr->n_obj[l];
  if (cand) for (int k = 0; k < S_NSTAGE; ++k) {
    cand[k] = s.h_hdr->cand[k];
    cand[S_NSTAGE + k] = s.h_hdr->cl_used[k];
    cand[2 * S_NSTAGE + k] = k == S_LS ? s.h_hdr->cand_eval[k] : s.h_hdr->cand[k];
  }
  return LST_OK;
}

static const uint32_t kArity[LST_NLEVEL] = {2, 4, 6, 10, 6, 10, 14};

extern "C" int lst_get_objects(lst_ctx *c, uint32_t slot, lst_level level, int copy_to_host, lst_objects *out) {
  if (!c || slot >= c->n_slots || !out || (int)level < 0 || level >= LST_NLEVEL) return einval();
  Slot &s = c->slots[slot];
  if (!s.ran) return LST_ESTATE;
  launch_export(c->k, s.dev, (int)level, s.last_stream);
  CU(cudaGetLastError());
  const int rc = sync_header(c, s);
  if (rc != LST_OK) return rc;
  lst_objects o;
  memset(&o, 0, sizeof(o));
  o.n = s.h_hdr->n_obj[level];
  o.arity = kArity[level];
  const uint8_t *keep_d = level == LST_T5 ? s.dev.t5_keep : level == LST_PT3 ? s.dev.pt3_keep
                          : level == LST_PT5 ? s.dev.pt5_keep : nullptr;
  if (!copy_to_host) {
    o.hit_idx = s.dev.exp_hits; o.parents = s.dev.exp_par; o.f = s.dev.exp_f; o.keep = keep_d; o.on_device = 1;
  } else {
    if (!s.h_hits) {
      CU(cudaMallocHost((void **)&s.h_hits, sizeof(uint32_t) * c->exp_hit_words));
      CU(cudaMallocHost((void **)&s.h_par, sizeof(uint32_t) * 2 * c->exp_obj_cap));
      CU(cudaMallocHost((void **)&s.h_f, sizeof(float) * 4 * c->exp_obj_cap));
      CU(cudaMallocHost((void **)&s.h_keep, c->exp_obj_cap));
    }
    if (o.n) {
      CU(cudaMemcpyAsync(s.h_hits, s.dev.exp_hits, sizeof(uint32_t) * (size_t)o.n * o.arity, cudaMemcpyDeviceToHost, s.last_stream));
      CU(cudaMemcpyAsync(s.h_par, s.dev.exp_par, sizeof(uint32_t) * 2 * (size_t)o.n, cudaMemcpyDeviceToHost, s.last_stream));
      CU(cudaMemcpyAsync(s.h_f, s.dev.exp_f, sizeof(float) * 4 * (size_t)o.n, cudaMemcpyDeviceToHost, s.last_stream));
      if (keep_d) CU(cudaMemcpyAsync(s.h_keep, keep_d, o.n, cudaMemcpyDeviceToHost, s.last_stream));
      CU(cudaStreamSynchronize(s.last_stream));
    }
    o.hit_idx = s.h_hits; o.parents = s.h_par; o.f = s.h_f; o.keep = keep_d ? s.h_keep : nullptr; o.on_device = 0;
  }
  *out = o;
  return LST_OK;
}

extern "C" uint32_t lst_launches_per_run(const lst_ctx *c) { return c ? c->launches.load() : 0; }

// The chain without a graph, one CUDA event after every kernel; synchronises the stream.
extern "C" int lst_run_timed(lst_ctx *c, uint32_t slot, void *cuda_stream, uint32_t max_kernels, const char **names,
                             float *ms, uint32_t *n_kernels) {
  if (!c || slot >= c->n_slots || !n_kernels) return einval();
  Slot &s = c->slots[slot];
  if (!s.bound || !s.loaded) return LST_ESTATE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (!s.timed) {
    s.timed = new (std::nothrow) Recorder();
    if (!s.timed) return LST_ENOMEM;
    for (int k = 0; k <= Recorder::kMax; ++k) CU(cudaEventCreate(&s.timed->ev[k]));
  }
  Recorder &r = *s.timed;
  r.timed = true;
  r.n = 0;
  CU(cudaEventRecord(r.ev[0], st));
  c->launches.store((uint32_t)enqueue_chain(c, slot, 1, st, &r, false));
  CU(cudaGetLastError());
  s.ran = true; s.last_stream = st;
  CU(cudaStreamSynchronize(st));
  const uint32_t n = std::min<uint32_t>((uint32_t)r.n, max_kernels);
  for (uint32_t k = 0; k < n; ++k) {
    float t = 0.f;
    CU(cudaEventElapsedTime(&t, r.ev[k], r.ev[k + 1]));
    if (ms) ms[k] = t;
    if (names) names[k] = r.name[k];
  }
  *n_kernels = (uint32_t)r.n;
  return LST_OK;
}

// ------------------------------------------------------------------ host test hooks (include/lst_test.h)
// Run the very same __host__ __device__ selection arithmetic on the CPU (tests only; no GPU needed).
extern "C" int lst_host_eval(const lst_config *cfg_in, int level, uint32_t n, const float *pts, const uint8_t *cats,
                             const double *aux, uint8_t *pass, uint8_t *pre, double *f) {
  lst_config cfg;
  if (cfg_in) cfg = *cfg_in; else lst_default_config(&cfg);
  Params g;
  make_params(cfg, &g);
  const int npts = level == LST_MD ? 2 : level == LST_LS ? 2 : level == LST_T3 ? 3 : level == LST_T5 ? 5 : 0;
  if (!npts || !pts || !cats || !pass) return einval();
  for (uint32_t i = 0; i < n; ++i) {
    Pt P[5];
    const float *p = pts + (size_t)i * npts * 3;
    const uint8_t *ct = cats + (size_t)i * npts;
    for (int k = 0; k < npts; ++k) P[k] = make_pt(p[3 * k], p[3 * k + 1], p[3 * k + 2], ct[k]);
    double o3[3] = {0, 0, 0};
    bool ok = false, pr = true;
    if (level == LST_MD) {
      MdOut o = {0, 0, 0};
      ok = md_eval_d(g, P[0], P[1], ct[0], &o);
      const float rl = sqrtf(p[0] * p[0] + p[1] * p[1]), ru = sqrtf(p[3] * p[3] + p[4] * p[4]);
      pr = md_pre_f(g, p[0], p[1], p[2], rl, p[3], p[4], p[5], ru, ct[0]);
      o3[0] = o.kappa; o3[1] = o.sigk; o3[2] = o.dphi;
    } else if (level == LST_LS) {
      const double *a = aux + 4 * (size_t)i;
      LsOut o = {0, 0, 0};
      ok = ls_eval_d(g, P[0], a[0], a[1], P[1], a[2], a[3], &o);
      const float ri = sqrtf(p[0] * p[0] + p[1] * p[1]), ro = sqrtf(p[3] * p[3] + p[4] * p[4]);
      // what k_ls_eval applies: tier 1, then L3 in its mode-R form or the full mode-Z pre-filter
      pr = ls_tier1_f(g, p[0], p[1], p[2], ri, g.f_sig_z[ct[0]], g.f_sig_r[ct[0]], g.f_sig_t[ct[0]], p[3], p[4], p[5], ro,
                      g.f_sig_z[ct[1]], g.f_sig_r[ct[1]], g.f_sig_t[ct[1]], ct[1] >= 2) &&
           (ct[1] < 2 ? ls_l3_modeR_f(g, p[0], p[1], ri, (float)a[0], (float)a[1], g.f_sig_t[ct[0]], ct[0] >= 2, p[3], p[4], ro,
                                      (float)a[2], (float)a[3], g.f_sig_t[ct[1]])
                      : ls_pre_f(g, p[0], p[1], p[2], ri, (float)a[0], (float)a[1], ct[0], p[3], p[4], p[5], ro, (float)a[2],
                                 (float)a[3], ct[1]));
      o3[0] = o.kappa; o3[1] = o.sigk; o3[2] = o.dphi;
    } else if (level == LST_T3) {
      T3Out o = {0, 0, 0};
      ok = t3_eval_d(g, P[0], P[1], P[2], &o);
      pr = t3_pre_f(g, p[0], p[1], p[2], sqrtf(p[0] * p[0] + p[1] * p[1]), ct[0], p[3], p[4], p[5],
                    sqrtf(p[3] * p[3] + p[4] * p[4]), ct[1], p[6], p[7], p[8], sqrtf(p[6] * p[6] + p[7] * p[7]), ct[2]);
      o3[0] = o.kappa3; o3[1] = o.sigk3; o3[2] = o.beta;
    } else {
      const double *a = aux + 4 * (size_t)i;
      T5Out o = {0, 0, 0, 0, 0};
      ok = t5_eval_d(g, P, a[0], a[1], a[2], a[3], &o);
      o3[0] = o.R; o3[1] = o.chi2; o3[2] = o.eta;
    }
    pass[i] = ok;
    if (pre) pre[i] = pr;
    if (f) { f[3 * (size_t)i] = o3[0]; f[3 * (size_t)i + 1] = o3[1]; f[3 * (size_t)i + 2] = o3[2]; }
  }
  return LST_OK;
}

extern "C" int lst_host_ls_window(const lst_config *cfg_in, uint32_t n, const float *row, const uint8_t *row_cat,
                                  const float *box, const uint8_t *box_cat, uint8_t *live, float *w) {
  if (!row || !row_cat || !box || !box_cat || !live || !w) return einval();
  lst_config cfg;
  if (cfg_in) cfg = *cfg_in; else lst_default_config(&cfg);
  Params g;
  make_params(cfg, &g);
  for (uint32_t i = 0; i < n; ++i) {
    float ww = 4.0f;
    live[i] = ls_row_window(g, row[2 * i], row[2 * i + 1], row_cat[i] & 3, box[4 * i], box[4 * i + 1], box[4 * i + 2],
                            box[4 * i + 3], box_cat[i] & 3, &ww);
    w[i] = ww;
  }
  return LST_OK;
}

// Test hook (include/lst_test.h): what a0 left in the slot, copied to host arrays.  Reads only.
extern "C" int lst_test_get_hit_index(lst_ctx *c, uint32_t slot, uint32_t *det_off, uint32_t *hit_orig, float *hit_xyzr,
                                      uint32_t *n_hits_out) {
  if (!c || slot >= c->n_slots) return einval();
  Slot &s = c->slots[slot];
  if (!s.ran) return LST_ESTATE;
  const int rc = sync_header(c, s);
  if (rc != LST_OK) return rc;
  const uint32_t n = s.h_hdr->n_hits, n_det = c->k.geo.n_det;
  if (det_off) CU(cudaMemcpy(det_off, s.dev.det_off, sizeof(uint32_t) * ((size_t)n_det + 1), cudaMemcpyDeviceToHost));
  if (hit_orig && n) CU(cudaMemcpy(hit_orig, s.dev.hit_orig, sizeof(uint32_t) * (size_t)n, cudaMemcpyDeviceToHost));
  if (hit_xyzr && n) CU(cudaMemcpy(hit_xyzr, s.dev.hit, sizeof(float4) * (size_t)n, cudaMemcpyDeviceToHost));
  if (n_hits_out) *n_hits_out = n;
  return LST_OK;
}
