// k_t3t5.cu -- a3 triplets (Fig. 5, 8; reading C4) and a4 quintuplets (PAPER.md:73,
// Fig. 9; reading C5: radius match, middle triplet, weighted Kasa circle-fit chi2).
//
// Both are joins on a shared mini-doublet: a T3 is LS (1,2) + LS (2,3), a T5 is T3 (1,2,3) +
// T3 (3,4,5).  Left objects are the rows; the right list of a row is the contiguous range of
// objects whose first MD is the row's last MD (LS are grouped by inner MD, T3 by first MD).
// Groups are chunks of kRowChunk rows; a group's candidates are numbered row-major.
#include "lst_launch.h"

namespace lst {

struct RowTab {                       // right-list table of one group, in shared memory
  uint32_t start[kRowChunk];
  uint32_t cum[kRowChunk + 1];
  uint32_t hint[kItemWords];          // row of the item's candidates 0, 32, 64, ... (stage_hints)
};

// KIND 0 (T3) : rows are LS, right lists are LS ranges of the outer MD.
// KIND 1 (T5) : rows are T3, right lists are T3 ranges of the third MD.
// KIND 2 (pT5): rows are (seed, compatible start module) pairs (k_pix.cu), right lists are the T5
//               whose first MD lies in that module (T5 are ordered by first MD, MDs by module).
// KIND 3 (pT3): same with T3.
enum { J_T3 = 0, J_T5 = 1, J_PT5 = 2, J_PT3 = 3 };

template <int KIND> struct JoinTraits;
template <> struct JoinTraits<J_T3> {
  static constexpr const char *n_groups = "k_join_groups[T3]", *n_eval = "k_join_eval[T3]", *n_decide = "k_join_decide[T3]", *n_fill = "k_join_fill[T3]";
  static constexpr int stage = S_T3, rows_level = 1, out_level = 2; };
template <> struct JoinTraits<J_T5> {
  static constexpr const char *n_groups = "k_join_groups[T5]", *n_eval = "k_join_eval[T5]", *n_decide = "k_join_decide[T5]", *n_fill = "k_join_fill[T5]";
  static constexpr int stage = S_T5, rows_level = 2, out_level = 3; };
template <> struct JoinTraits<J_PT5> {
  static constexpr const char *n_groups = "k_join_groups[pT5]", *n_eval = "k_join_eval[pT5]", *n_decide = "k_join_decide[pT5]", *n_fill = "k_join_fill[pT5]";
  static constexpr int stage = S_PT5, rows_level = kPairLevel, out_level = 5; };
template <> struct JoinTraits<J_PT3> {
  static constexpr const char *n_groups = "k_join_groups[pT3]", *n_eval = "k_join_eval[pT3]", *n_decide = "k_join_decide[pT3]", *n_fill = "k_join_fill[pT3]";
  static constexpr int stage = S_PT3, rows_level = kPairLevel, out_level = 4; };

template <int KIND>
__device__ __forceinline__ void right_range(const SlotDev &s, uint32_t row, uint32_t *st, uint32_t *cnt) {
  if (KIND == J_T3) {
    const uint32_t mo = s.ls_md[row].y;
    *st = s.ls_md_off[mo];
    *cnt = s.ls_md_off[mo + 1] - *st;
  } else if (KIND == J_T5) {
    const uint32_t m3 = s.t3_md[row].z;
    *st = s.t3_md_off[m3];
    *cnt = s.t3_md_off[m3 + 1] - *st;
  } else {
    // objects whose first MD lies in the row's module AND inside the row's azimuthal window (the MD
    // range k_px_modules found: objects are grouped by first MD)
    const uint2 rng = s.px_rng[row];
    const uint32_t *off = KIND == J_PT5 ? s.t5_md_off : s.t3_md_off;
    *st = off[rng.x];
    *cnt = off[rng.y] - *st;
  }
}

template <int KIND>
__global__ void k_join_groups(SlotDev s) {
  const int stage = JoinTraits<KIND>::stage;
  const StageBuf &st = s.st[stage];
  const uint32_t n_rows = s.hdr->n_obj[JoinTraits<KIND>::rows_level];
  const uint32_t ng = (n_rows + kRowChunk - 1) / kRowChunk;
  const int lane = threadIdx.x & 31;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
  for (uint32_t gidx = warp; gidx < ng; gidx += nwarp) {
    const uint32_t r0 = gidx * kRowChunk, r1 = min(r0 + kRowChunk, n_rows);
    uint32_t sum = 0;
    for (uint32_t r = r0 + lane; r < r1; r += 32) {
      uint32_t a, c;
      right_range<KIND>(s, r, &a, &c);
      sum += c;
    }
    sum = warp_sum(sum);
    if (lane == 0) { st.gR[gidx] = 1; st.gW[gidx] = sum; }
  }
}

template <int KIND>
__device__ __forceinline__ void stage_rows(RowTab &rt, const SlotDev &s, uint32_t r0, uint32_t n_rows, uint32_t *sh) {
  const int tid = threadIdx.x;   // kThreads == kRowChunk
  uint32_t a = 0, c = 0;
  if (r0 + tid < n_rows) right_range<KIND>(s, r0 + tid, &a, &c);
  uint32_t tot;
  const uint32_t e = block_excl_scan(c, sh, &tot);
  rt.start[tid] = a;
  rt.cum[tid] = e;
  if (tid == 0) rt.cum[kRowChunk] = tot;
  __syncthreads();
}
// flat candidate -> (row in group, right object)
__device__ __forceinline__ void flat_to_pair(const RowTab &rt, uint32_t cf, int *row, uint32_t *right) {
  int lo = 0, hi = kRowChunk;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (rt.cum[mid] <= cf) lo = mid; else hi = mid;
  }
  *row = lo;
  *right = rt.start[lo] + (cf - rt.cum[lo]);
}

// Per item: the row of every 32nd candidate, so that a candidate finds its row by a short linear
// walk (rows are ~100 candidates wide) instead of a 7-step binary search.
__device__ __forceinline__ void stage_hints(RowTab &rt, uint32_t j0) {
  if (threadIdx.x < kItemWords) {
    const uint32_t cf = j0 + 32u * threadIdx.x;
    int row = 0;
    if (cf < rt.cum[kRowChunk]) { uint32_t b; flat_to_pair(rt, cf, &row, &b); }
    rt.hint[threadIdx.x] = (uint32_t)row;
  }
  __syncthreads();
}
// candidate c of the item (flat index cf = j0 + c < total) -> (row in group, right object)
__device__ __forceinline__ void item_to_pair(const RowTab &rt, uint32_t j0, int c, int *row, uint32_t *right) {
  const uint32_t cf = j0 + (uint32_t)c;
  int r = (int)rt.hint[c >> 5];
  while (rt.cum[r + 1] <= cf) ++r;
  *row = r;
  *right = rt.start[r] + (cf - rt.cum[r]);
}

__device__ __forceinline__ Pt md_point(const SlotDev &s, uint32_t md) {
  const float4 p = s.md_pos[md];
  return make_pt(p.x, p.y, p.z, (int)(s.md_mod[md] & 3u));
}

// ------------------------------------------------------------------ evaluation of one candidate
__device__ __forceinline__ bool t3_candidate(const SlotDev &s, const Params &g, uint32_t a, uint32_t b, T3Out *o,
                                             uint4 *mds) {
  const uint2 la = s.ls_md[a], lb = s.ls_md[b];
  const Pt P1 = md_point(s, la.x), P2 = md_point(s, la.y), P3 = md_point(s, lb.y);
  if (mds) *mds = make_uint4(la.x, la.y, lb.y, 0u);
  return t3_eval_d(g, P1, P2, P3, o);
}
__device__ __forceinline__ bool t5_candidate(const SlotDev &s, const Params &g, uint32_t a, uint32_t b, T5Out *o,
                                             uint32_t *mds, double2 *ka, double2 *kb) {
  const double2 k3a = s.t3_kd[a], k3b = s.t3_kd[b];
  if (ka) { *ka = k3a; *kb = k3b; }
  if (!o && !le(fabs(k3a.x - k3b.x), g.ns * (k3a.y + k3b.y))) return false;   // early T5-1
  const uint4 ta = s.t3_md[a], tb = s.t3_md[b];
  const uint32_t m[5] = {ta.x, ta.y, ta.z, tb.y, tb.z};
  Pt P[5];
#pragma unroll
  for (int k = 0; k < 5; ++k) { P[k] = md_point(s, m[k]); if (mds) mds[k] = m[k]; }
  return t5_eval_d(g, P, k3a.x, k3a.y, k3b.x, k3b.y, o);
}

// pT5 / pT3 candidate: pixel seed against OT object `obj` (reading C6).  The fp32 pre-filter tests
// the first and the last anchor, loosened by kPreSlack plus absolute slacks far above the fp32 error
// (1e-5 rad on a >= 4e-3 rad window, 2e-3 cm on a >= 0.2 cm window); it never rejects on NaN.
// sp = {kappa_p, sinh eta, phi, z0} of the seed, computed once per row (stage_seeds).
// one anchor (MD m) against the seed parameters sp
__device__ __forceinline__ bool px_anchor_f(const SlotDev &s, const Params &g, float4 sp, uint32_t m) {
  const float4 h = s.md_pos[m];
  const int cat = (int)(s.md_mod[m] & 3u);
  const float kp = sp.x, sh = sp.y;
  float al;
  if (cat < 2) {
    const float kr = kp * h.w;
    al = fabsf(kr) <= 1e-4f ? h.w : __fdividef(asinf(fminf(1.0f, fmaxf(-1.0f, kr))), kp);
  } else {
    al = __fdividef(h.z - sp.w, sh);
  }
  const float d = s.md_phi[m] - (sp.z + kp * al);
  const float dph = d - 6.2831853071795864769f * rintf(d * 0.15915494309189533577f);
  const float sgp = (float)g.seed_sig_phi + (float)g.seed_sig_pt * fabsf(kp) * al + __fdividef(g.f_sig_t[cat], h.w);
  if (fabsf(dph) > g.f_ns * sgp * kPreSlack + 1e-5f) return false;
  float dzt, szt;
  if (cat < 2) {
    dzt = h.z - (sp.w + sh * al);
    szt = (float)g.seed_sig_z + g.f_sig_z[cat];
  } else {
    const float ka = kp * al;
    dzt = h.w - (fabsf(ka) <= 1e-4f ? al : __fdividef(sinf(ka), kp));
    szt = __fdividef((float)g.seed_sig_z, fabsf(sh)) + g.f_sig_r[cat];
  }
  if (fabsf(dzt) > g.f_ns * szt * kPreSlack + 2e-3f) return false;
  return true;
}
// first and last anchor of the object (the last one has the longest lever arm: together they leave
// the fp64 kernel little more than the accepted pairs)
template <int KIND>
__device__ __forceinline__ bool px_pre_f(const SlotDev &s, const Params &g, float4 sp, uint32_t obj) {
  uint32_t m0, m1;
  if (KIND == J_PT5) { m0 = s.t5_md[5 * (size_t)obj]; m1 = s.t5_md[5 * (size_t)obj + 4]; }
  else { const uint4 t = s.t3_md[obj]; m0 = t.x; m1 = t.z; }
  return px_anchor_f(s, g, sp, m0) && px_anchor_f(s, g, sp, m1);
}

// fp64 decision (and chi2_pix) of one (seed, object) pair.
template <int KIND>
__device__ __forceinline__ bool px_candidate(const GeoDev &geo, const SlotDev &s, const Params &g, uint32_t p,
                                             uint32_t obj, double *chi2) {
  constexpr int N = KIND == J_PT5 ? 5 : 3;
  uint32_t m[5];
  if (KIND == J_PT5) {
#pragma unroll
    for (int k = 0; k < 5; ++k) m[k] = s.t5_md[5 * (size_t)obj + k];
  } else {
    const uint4 t = s.t3_md[obj];
    m[0] = t.x; m[1] = t.y; m[2] = t.z;
  }
  Seed sd;
  sd.pt = (double)s.seed_pt[p]; sd.eta = (double)s.seed_eta[p]; sd.phi = (double)s.seed_phi[p];
  sd.z0 = (double)s.seed_z0[p]; sd.q = s.seed_q[p];
  Pt P[N];
#pragma unroll
  for (int k = 0; k < N; ++k) P[k] = md_point(s, m[k]);
  double c2 = 0.0;
  const bool ok = px_eval_d(g, sd, P, N, (int)geo.layer[s.md_mod[m[0]] >> 2], &c2);
  if (chi2) *chi2 = c2;
  return ok;
}

// per-row seed parameters of the pixel joins: {kappa_p, sinh eta, phi, z0}
__device__ __forceinline__ void stage_seeds(float4 *rowseed, const SlotDev &s, const Params &g, uint32_t r0,
                                            uint32_t n_rows) {
  const int tid = threadIdx.x;   // kThreads == kRowChunk
  float4 v = make_float4(0.f, 1.f, 0.f, 0.f);
  if (r0 + tid < n_rows) {
    const uint32_t p = s.px_pair[r0 + tid].x;
    v.x = -(float)s.seed_q[p] * (float)g.kB / (2.0f * s.seed_pt[p]);
    v.y = sinhf(s.seed_eta[p]);
    v.z = s.seed_phi[p];
    v.w = s.seed_z0[p];
  }
  rowseed[tid] = v;
}

// Phase 1 of a join candidate: a cheap necessary condition evaluated on every candidate (T3: the
// fp32 pre-filter t3_pre_f; T5: the radius match T5-1 on the stored kappa3; pixel: the fp32
// first-anchor pre-filter).  *ab = the pair handed to the decide kernel.
template <int KIND>
__device__ __forceinline__ bool join_phase1(const SlotDev &s, const Params &g, uint32_t row, uint32_t b,
                                            const float4 *rowseed, int lrow, uint2 *ab) {
  *ab = make_uint2(row, b);
  if (KIND == J_T3) {
    const uint2 la = s.ls_md[row], lb = s.ls_md[b];
    const float4 p1 = s.md_pos[la.x], p2 = s.md_pos[la.y], p3 = s.md_pos[lb.y];
    const int c1 = (int)(s.md_mod[la.x] & 3u), c2 = (int)(s.md_mod[la.y] & 3u), c3 = (int)(s.md_mod[lb.y] & 3u);
    return t3_pre_f(g, p1.x, p1.y, p1.z, p1.w, c1, p2.x, p2.y, p2.z, p2.w, c2, p3.x, p3.y, p3.z, p3.w, c3);
  }
  if (KIND == J_T5) {
    const double2 k3a = s.t3_kd[row], k3b = s.t3_kd[b];
    if (!le(fabs(k3a.x - k3b.x), g.ns * (k3a.y + k3b.y))) return false;          // T5-1 (exact, fp64)
    // T5-2: the middle triplet (MD 2, 3, 4) through the fp32 triplet pre-filter
    const uint4 ta = s.t3_md[row], tb = s.t3_md[b];
    const float4 p2 = s.md_pos[ta.y], p3 = s.md_pos[ta.z], p4 = s.md_pos[tb.y];
    const int c2 = (int)(s.md_mod[ta.y] & 3u), c3 = (int)(s.md_mod[ta.z] & 3u), c4 = (int)(s.md_mod[tb.y] & 3u);
    return t3_pre_f(g, p2.x, p2.y, p2.z, p2.w, c2, p3.x, p3.y, p3.z, p3.w, c3, p4.x, p4.y, p4.z, p4.w, c4);
  }
  ab->x = s.px_pair[row].x;     // the seed
  return px_pre_f<KIND>(s, g, rowseed[lrow], b);
}

// Pre-filter kernel: every candidate of every item through phase 1; survivors go to the stage's
// candidate list.  One barrier-free candidate loop per item after the row table is staged.
template <int KIND>
__global__ void __launch_bounds__(kThreads) k_join_eval(GeoDev geo, SlotDev s, Params g) {
  __shared__ RowTab rt;
  __shared__ uint32_t sh[33];
  __shared__ float4 rowseed[(KIND == J_PT5 || KIND == J_PT3) ? kRowChunk : 1];
  __shared__ ClStageT<64> cl_mem[kThreads / 32];
  (void)geo;
  ClBufT<64> cl;
  cl.init(&cl_mem[threadIdx.x >> 5]);
  const int stage = JoinTraits<KIND>::stage;
  const StageBuf &st = s.st[stage];
  const uint32_t n_items = s.hdr->n_items[stage];
  const uint32_t n_rows = s.hdr->n_obj[JoinTraits<KIND>::rows_level];
  const int tid = threadIdx.x;
  // The pixel stages have few items (~700) and a latency-bound candidate loop: an item is split over
  // kSplit blocks (each stages the rows and takes a quarter of the candidates).
  constexpr uint32_t kSplit = (KIND == J_PT5 || KIND == J_PT3) ? 4u : 1u;
  constexpr int kPart = kItemCand / (int)kSplit;
  for (uint32_t v = blockIdx.x; v < n_items * kSplit; v += gridDim.x) {
    const uint32_t it = v / kSplit, part = v % kSplit;
    const Item item = st.items[it];
    if (part != 0 && (int)(part * kPart) >= (int)item.nj) continue;      // uniform per block
    const uint32_t r0 = item.group * kRowChunk;
    const uint32_t key0 = it * (uint32_t)kItemCand;
    if (part == 0 && tid < kItemWords) st.mask[(size_t)it * kItemWords + tid] = 0;   // the decide kernel ORs the pass bits in
    if (KIND == J_PT5 || KIND == J_PT3) stage_seeds(rowseed, s, g, r0, n_rows);
    stage_rows<KIND>(rt, s, r0, n_rows, sh);
    stage_hints(rt, item.j0);
    const int nj = min((int)item.nj, (int)((part + 1) * kPart));
    for (int base = (int)(part * kPart); base < nj; base += kThreads) {
      const int c = base + tid;
      bool keep = false;
      uint2 ab = make_uint2(0u, 0u);
      if (c < nj) {
        int row; uint32_t b;
        item_to_pair(rt, item.j0, c, &row, &b);
        keep = join_phase1<KIND>(s, g, r0 + row, b, rowseed, row, &ab);
      }
      cl.push(s.hdr, st, stage, keep, key0 + (uint32_t)c, ab);
    }
    __syncthreads();
  }
  cl.flush_all(s.hdr, st, stage);
}

// Decide kernel: the fp64 decision of the listed candidates, one thread each (dense warps, no
// staging); an accepted candidate sets its pass bit and writes its results to the stage's pool.
template <int KIND>
__global__ void __launch_bounds__(128) k_join_decide(GeoDev geo, SlotDev s, Params g) {
  const int stage = JoinTraits<KIND>::stage;
  const StageBuf &st = s.st[stage];
  Header *hdr = s.hdr;
  const uint32_t n = min(hdr->cl_used[stage], st.cap_cl);
  const uint32_t nround = (n + 31u) & ~31u;
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < nround; j += gridDim.x * blockDim.x) {
    const bool live = j < n;
    const uint32_t key = live ? st.cl_key[j] : 0u;
    const uint2 ab = live ? st.cl_ab[j] : make_uint2(0u, 0u);
    bool pass = false;
    if (KIND == J_T3) {
      T3Out o;
      if (live) pass = t3_candidate(s, g, ab.x, ab.y, &o, nullptr);
      if (pass) {
        st.p_d2[j] = make_double2(o.kappa3, o.sigk3);
        st.p_f4[j] = make_float4((float)o.beta, 0.f, 0.f, 0.f);
      }
    } else if (KIND == J_T5) {
      T5Out o;
      if (live) pass = t5_candidate(s, g, ab.x, ab.y, &o, nullptr, nullptr, nullptr);
      if (pass) {
        st.p_d2[j] = make_double2(o.eta, o.phi);
        st.p_d2b[j] = make_double2(o.chi2, o.R);
        st.p_f4[j] = make_float4((float)o.pt, 0.f, 0.f, 0.f);
      }
    } else {
      double c2 = 0.0;
      if (live) pass = px_candidate<KIND>(geo, s, g, ab.x, ab.y, &c2);
      if (pass) st.p_d2[j] = make_double2(c2, 0.0);
    }
    if (pass) atomicOr(&st.mask[(size_t)(key / kItemCand) * kItemWords + ((key % kItemCand) >> 5)], 1u << (key & 31u));
  }
}

// One thread per pool entry: canonical position; constituent indices re-read from the inputs.
template <int KIND>
__global__ void __launch_bounds__(256) k_join_fill(SlotDev s) {
  const int stage = JoinTraits<KIND>::stage;
  const StageBuf &st = s.st[stage];
  const Header *hdr = s.hdr;
  if (hdr->n_obj[JoinTraits<KIND>::out_level] == 0) return;
  const uint32_t n = min(hdr->cl_used[stage], st.cap_cl);
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
    const uint32_t idx = pool_target(st, st.cl_key[j]);
    if (idx == 0xFFFFFFFFu) continue;
    const uint2 ab = st.cl_ab[j];
    if (KIND == J_T3) {
      const uint2 la = s.ls_md[ab.x], lb = s.ls_md[ab.y];
      s.t3_md[idx] = make_uint4(la.x, la.y, lb.y, 0u);
      s.t3_ls[idx] = ab;
      s.t3_kd[idx] = st.p_d2[j];
      s.t3_beta[idx] = st.p_f4[j].x;
    } else if (KIND == J_T5) {
      const uint4 ta = s.t3_md[ab.x], tb = s.t3_md[ab.y];
      const uint32_t m[5] = {ta.x, ta.y, ta.z, tb.y, tb.z};
#pragma unroll
      for (int q = 0; q < 5; ++q) s.t5_md[(size_t)5 * idx + q] = m[q];
      const double2 cr = st.p_d2b[j];
      s.t5_t3[idx] = ab;
      s.t5_chi2[idx] = cr.x;
      s.t5_etaphi[idx] = st.p_d2[j];
      s.t5_f[idx] = make_float4((float)cr.y, (float)cr.x, (float)s.t3_kd[ab.x].x, (float)s.t3_kd[ab.y].x);
      s.t5_pt[idx] = st.p_f4[j].x;
    } else if (KIND == J_PT5) {
      s.pt5_po[idx] = ab; s.pt5_chi2[idx] = st.p_d2[j].x;
    } else {
      s.pt3_po[idx] = ab; s.pt3_chi2[idx] = st.p_d2[j].x;
    }
  }
}

// ------------------------------------------------------------------ launchers
template <int KIND>
static void launch_join_t(const Ctx &c, const SlotDev &s, uint32_t row_cap, uint32_t out_cap, cudaStream_t st) {
  const int gg = (int)((row_cap / kRowChunk + 1 + 3) / 4);   // 4 warps per block, one group per warp
  k_join_groups<KIND><<<gg < c.n_sm * 8 ? gg : c.n_sm * 8, 128, 0, st>>>(s); LST_MARK(c, st, JoinTraits<KIND>::n_groups);
  launch_emit(c, s, JoinTraits<KIND>::stage, JoinTraits<KIND>::rows_level, st);
  k_join_eval<KIND><<<c.n_sm * 16, kThreads, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, JoinTraits<KIND>::n_eval);
  k_join_decide<KIND><<<c.n_sm * 4, 128, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, JoinTraits<KIND>::n_decide);
  launch_item_counts(c, s, JoinTraits<KIND>::stage, st);
  launch_scan_items(c, s, JoinTraits<KIND>::stage, JoinTraits<KIND>::out_level, out_cap, st);
  k_join_fill<KIND><<<c.n_sm * 4, 256, 0, st>>>(s); LST_MARK(c, st, JoinTraits<KIND>::n_fill);
}

void launch_join(const Ctx &c, const SlotDev &s, int kind, cudaStream_t st) {
  switch (kind) {
    case J_T3: launch_join_t<J_T3>(c, s, s.cap_ls, s.cap_t3, st); break;
    case J_T5: launch_join_t<J_T5>(c, s, s.cap_t3, s.cap_t5, st); break;
    case J_PT5: launch_join_t<J_PT5>(c, s, s.cap_seeds * kPxCap, s.cap_pt5, st); break;
    default: launch_join_t<J_PT3>(c, s, s.cap_seeds * kPxCap, s.cap_pt3, st); break;
  }
}

void launch_t3(const Ctx &c, const SlotDev &s, cudaStream_t st) {
  launch_join(c, s, J_T3, st);
  launch_row_offsets(c, s, 2, st);
}

void launch_t5(const Ctx &c, const SlotDev &s, cudaStream_t st) {
  launch_join(c, s, J_T5, st);
  launch_row_offsets(c, s, 3, st);
}

}  // namespace lst
