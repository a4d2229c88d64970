// k_mdls.cu -- a1 mini-doublets (Fig. 2; reading C1) and a2 line segments
// (Fig. 4-7; reading C3).
#include "lst_launch.h"

namespace lst {

// =================================================================== MD
// Work item = (module, rows of lower hits, columns of upper hits), <= 1024 pairs (typically ~100).
// k_md_eval: one THREAD per row (lower-sensor hit), walking the upper-sensor hits of its module: a
// module holds ~9 x 9 pairs, so per-module set-up by a warp cost more than the pairs themselves; every
// pair goes through the fp32 pre-filter, the survivors are appended to the stage's candidate list.  The
// row that starts a work item clears its pass bits (the decide kernel ORs them in).
// k_md_decide: one thread per listed pair, fp64 decision; accepted pairs set their pass bit and
// write kappa, sigma_kappa and dphi to the pool.
__global__ void __launch_bounds__(256) k_md_eval(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B,
                                                  const __grid_constant__ Params g) {
  __shared__ ClStageT<64> cl_mem[256 / 32];
  pdl_enter();
  LST_SLOT(B);
  const StageBuf &st = s.st[S_MD];
  const bool live = s.hdr->n_items[S_MD] != 0;      // 0: nothing to do, or the work list overflowed
  ClBufT<64> cl;
  cl.init(&cl_mem[threadIdx.x >> 5]);
  const uint32_t n_rows = live ? s.md_row0[geo.n_modules] : 0u;
  const uint32_t n_round = (n_rows + 31u) & ~31u;   // whole warps: the list appends are warp-cooperative
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < n_round; t += gridDim.x * blockDim.x) {
    uint32_t W = 0, hl = 0, up_m = 0, key0 = 0;
    int cat = 0;
    if (t < n_rows) {
      const uint32_t m = s.row_mod[t], r = t - s.md_row0[m];
      W = st.gW[m];
      cat = geo.category[m];
      hl = s.det_off[2 * m] + r;
      up_m = s.det_off[2 * m + 1];
      if (W) {
        uint32_t it, n_clear;
        if (W <= (uint32_t)kItemCand) {
          const uint32_t rpi = item_rpi(W), q = r / rpi;
          it = st.g_item0[m] + q;
          key0 = it * (uint32_t)kItemCand + (r - q * rpi) * W;
          n_clear = r == q * rpi ? 1u : 0u;
        } else {
          n_clear = item_nct(W);
          it = st.g_item0[m] + r * n_clear;
          key0 = it * (uint32_t)kItemCand;
        }
        for (uint32_t k = 0; k < n_clear; ++k) {
          uint4 *mw = reinterpret_cast<uint4 *>(st.mask + (size_t)(it + k) * kItemWords);
#pragma unroll
          for (int q4 = 0; q4 < kItemWords / 4; ++q4) mw[q4] = make_uint4(0u, 0u, 0u, 0u);
          st.item_group[it + k] = m;
        }
      }
    }
    const float4 l = s.hit[hl];
    const uint32_t Wmax = __reduce_max_sync(0xffffffffu, W);
    for (uint32_t j = 0; j < Wmax; ++j) {
      bool keep = false;
      const uint32_t hu = up_m + j;
      if (j < W) {
        const float4 u = s.hit[hu];
        keep = md_pre_f(g, l.x, l.y, l.z, l.w, u.x, u.y, u.z, u.w, cat);
      }
      // W > kItemCand: the row's candidates continue in the next item(s): key0 + j still addresses (item + j / 1024, j % 1024)
      cl.push(s.hdr, st, S_MD, keep, key0 + j, make_uint2(hl, hu));
    }
  }
  cl.flush_all(s.hdr, st, S_MD);
}

__global__ void __launch_bounds__(128) k_md_decide(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B,
                                                    const __grid_constant__ Params g) {
  pdl_enter();
  LST_SLOT(B);
  const StageBuf &st = s.st[S_MD];
  Header *hdr = s.hdr;
  const uint32_t n = min(hdr->cl_used[S_MD], st.cap_cl);
  const uint32_t nround = (n + 31u) & ~31u;
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < nround; j += gridDim.x * blockDim.x) {
    bool pass = false;
    MdOut o;
    uint32_t key = 0;
    if (j < n) {
      key = st.cl_key[j];
      const uint2 ab = st.cl_ab[j];
      const int cat = geo.category[st.item_group[key / kItemCand]];
      const float4 l = s.hit[ab.x], u = s.hit[ab.y];
      const Pt pl = make_pt(l.x, l.y, l.z, cat), pu = make_pt(u.x, u.y, u.z, cat);
      pass = md_eval_d(g, pl, pu, cat, &o);
    }
    if (pass) {
      atomicOr(&st.mask[(size_t)(key / kItemCand) * kItemWords + ((key % kItemCand) >> 5)], 1u << (key & 31u));
      st.p_d2[j] = make_double2(o.kappa, o.sigk);
      st.p_f4[j] = make_float4((float)o.dphi, 0.f, 0.f, 0.f);
    }
  }
}

// One thread per listed pair: the accepted ones move to their canonical position.  Then the MD range
// of every module (md_mod_off) from the rank of the module's first candidate.
__global__ void __launch_bounds__(256) k_md_fill(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B) {
  pdl_enter();
  LST_SLOT(B);
  const StageBuf &st = s.st[S_MD];
  const Header *hdr = s.hdr;
  const uint32_t n_md = hdr->n_obj[0], n_items = hdr->n_items[S_MD];
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nt = gridDim.x * blockDim.x;
  for (uint32_t m = tid; m <= geo.n_modules; m += nt)
    s.md_mod_off[m] = rank_before(st, n_items, n_md, st.g_item0[m] * (uint32_t)kItemCand);
  const uint32_t n = n_md ? min(hdr->cl_used[S_MD], st.cap_cl) : 0u;     // n_md == 0: nothing built, or overflow (level emptied)
  for (uint32_t j = tid; j < n; j += nt) {
    const uint32_t key = st.cl_key[j];
    const uint32_t idx = pool_target(st, key);
    if (idx == 0xFFFFFFFFu) continue;
    const uint32_t m = st.item_group[key / kItemCand];
    const uint2 h = st.cl_ab[j];
    const float4 l = s.hit[h.x];
    const double2 kd = st.p_d2[j];
    s.md_pos[idx] = l;
    s.md_kd[idx] = kd;
    s.md_kf[idx] = make_float2((float)kd.x, (float)kd.y);
    s.md_hit[idx] = h;
    s.md_mod[idx] = (m << 2) | (uint32_t)geo.category[m];
    st_f(s, s.md_dphi, idx, st.p_f4[j].x);
    s.md_phi[idx] = atan2f(l.y, l.x);
    s.md_prel[idx] = s.hit_key[h.x];
  }
}

// =================================================================== LS
// Group of module A: rows = MDs of A, width W_A = number of MDs in the modules connected to A (the
// candidates of the method's definition: all MD pairs in map-connected modules; a candidate's pass
// bit sits at (row, column) of that rectangle whatever part of it the enumeration visits).  The same
// warp also writes A's ModEv record for the per-row windows of k_ls_eval.
constexpr int kLsGroupWarps = 8;     // modules per block of k_ls_groups
__global__ void __launch_bounds__(32 * kLsGroupWarps) k_ls_groups(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B) {
  __shared__ uint32_t sh_items[kLsGroupWarps];
  __shared__ unsigned long long sh_cand[kLsGroupWarps];
  __shared__ uint32_t sh[33];
  pdl_enter();
  LST_SLOT(B);
  const StageBuf &st = s.st[S_LS];
  Header *hdr = s.hdr;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const uint32_t A = blockIdx.x * kLsGroupWarps + wib;
  uint32_t my_items = 0;
  unsigned long long my_cand = 0;
  if (A < geo.n_modules) {
    const uint32_t m0 = s.md_mod_off[A], R = s.md_mod_off[A + 1] - m0;
    uint32_t W = 0;
    float rlo = 3.0e38f, rhi = -3.0e38f, zlo = 3.0e38f, zhi = -3.0e38f;
    float pmin = 0.0f, inv_w = 0.0f;
    uint32_t edge_cnt = 0;
    if (R) {
      // the column of A's candidate rectangle at which each connected module's MDs start
      const uint32_t e0 = geo.map_off[A], e1 = geo.map_off[A + 1];
      for (uint32_t eb = e0; eb < e1; eb += 32) {
        const uint32_t e = eb + lane;
        uint32_t n = 0;
        if (e < e1) { const uint32_t mb = geo.map_cols[e]; n = s.md_mod_off[mb + 1] - s.md_mod_off[mb]; }
        uint32_t tot;
        const uint32_t ex = warp_excl_scan(n, &tot);
        if (e < e1) s.edge_col0[e] = W + ex;
        W += tot;
      }
      for (uint32_t k = lane; k < R; k += 32) {
        const float4 p = s.md_pos[m0 + k];
        rlo = fminf(rlo, p.w); rhi = fmaxf(rhi, p.w); zlo = fminf(zlo, p.z); zhi = fmaxf(zhi, p.z);
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        rlo = fminf(rlo, __shfl_xor_sync(0xffffffffu, rlo, o)); rhi = fmaxf(rhi, __shfl_xor_sync(0xffffffffu, rhi, o));
        zlo = fminf(zlo, __shfl_xor_sync(0xffffffffu, zlo, o)); zhi = fmaxf(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
      }
      // keys ascend inside a module: lane j counts the MDs below edge j + 1 of kModBins equal bins
      pmin = s.md_prel[m0];
      const float span = s.md_prel[m0 + R - 1] - pmin;
      if (R <= 0xFFFFu && span > 1e-6f) {
        inv_w = (float)kModBins / span;
        if (lane < kModBins - 1) {
          const float edge = pmin + (float)(lane + 1) * (span * (1.0f / (float)kModBins));
          uint32_t x = m0, y = m0 + R;
          while (x < y) { const uint32_t mid = (x + y) >> 1; if (s.md_prel[mid] < edge) x = mid + 1; else y = mid; }
          edge_cnt = x - m0;
        }
      }
    }
    // assemble the record: lanes 0 .. 13 hold the 14 counts
    const uint32_t c_even = __shfl_sync(0xffffffffu, edge_cnt, (2 * lane) & 31), c_odd = __shfl_sync(0xffffffffu, edge_cnt, (2 * lane + 1) & 31);
    uint32_t word = 0;
    if (lane == 0) word = __float_as_uint(rlo);
    else if (lane == 1) word = __float_as_uint(rhi);
    else if (lane == 2) word = __float_as_uint(zlo);
    else if (lane == 3) word = __float_as_uint(zhi);
    else if (lane == 4) word = __float_as_uint(pmin);
    else if (lane == 5) word = __float_as_uint(inv_w);
    else if (lane == 6) word = __float_as_uint(geo.phic[A]);
    else if (lane == 7) word = m0;
    else if (lane == 8) word = R | ((uint32_t)geo.category[A] << 30);
    if (lane < 7) {   // words 9 .. 15 = cum[0 .. 13]
      const uint32_t packed = (c_even & 0xFFFFu) | (c_odd << 16);
      reinterpret_cast<uint32_t *>(&s.mod_ev[A])[9 + lane] = packed;
    }
    if (lane < 9) reinterpret_cast<uint32_t *>(&s.mod_ev[A])[lane] = word;
    if (lane == 0) {
      st.gR[A] = R;
      st.gW[A] = W;
    }
    my_items = items_of(R, W);
    my_cand = (unsigned long long)R * W;
  }
  // first item of every group: exclusive prefix inside the block here, across blocks in the last block
  if (lane == 0) { sh_items[wib] = my_items; sh_cand[wib] = my_cand; }
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t acc = 0;
    unsigned long long cs = 0;
    for (int k = 0; k < kLsGroupWarps; ++k) {
      const uint32_t g = blockIdx.x * kLsGroupWarps + k;
      if (g < geo.n_modules) st.g_item0[g] = acc;
      acc += sh_items[k]; cs += sh_cand[k];
    }
    st.gblk[blockIdx.x] = acc;
    if (cs) atomicAdd(&hdr->cand[S_LS], cs);
  }
  if (!last_block(&hdr->ticket[TK_GROUPS + S_LS], gridDim.x)) return;
  const uint32_t total = lb_scan_parts(st.gblk, gridDim.x, sh);
  const uint32_t ng = geo.n_modules;
  lb_add_block_prefix(st.g_item0, ng, st.gblk, kLsGroupWarps);
  if (threadIdx.x == 0) {
    const bool overflow = total > st.cap_items;
    st.g_item0[ng] = total;
    hdr->n_groups[S_LS] = ng;
    hdr->n_items[S_LS] = overflow ? 0u : total;
    if (overflow) atomicOr(&hdr->err, (uint32_t)ERR_CAP_ITEMS);
  }
}


// k_ls_eval: the fp32 pre-filter of the LS stage.  A warp takes kLsGrab consecutive rows (inner MDs)
// at a time, handed out dynamically.  The definition is "all MDs of the modules connected to the
// row's module"; the enumeration visits only the MDs that can pass cuts L1 / L2 for THAT row:
//   * the (row, connected module) pairs of the grabbed rows are flattened over the lanes; a lane tests
//     the box of its module's MD anchors against its row's pointing cone (L1) and azimuthal window
//     (L2), ls_row_window, and turns the window into an index range of the module's MDs (they ascend
//     in azimuth) through the bin counts of the module's ModEv record: no search, one 64-byte load;
//   * the ranges of 32 pairs are flattened again: lane c takes candidate c of their concatenation
//     (its segment = number of segment starts <= c, from one __reduce_or_sync of the start bits);
//   * tier 1 (ls_tier1_f; for an outer MD in a barrel module also L3, ls_l3_modeR_f) on every visited
//     candidate; mode-R survivors go straight to the stage's candidate list, mode-Z survivors
//     through a warp queue to ls_pre_f on 32 dense lanes.
// A candidate's key is that of the full rectangle: key_base(row) + column index in the row's column list.
constexpr int kLsGrab = 4;
// key of the first candidate of row r (relative to its module A, W > 0 columns) and the items the row starts
__device__ __forceinline__ uint32_t ls_key_base(const StageBuf &st, uint32_t A, uint32_t r, uint32_t W, uint32_t *first_item,
                                                uint32_t *n_start) {
  if (W <= (uint32_t)kItemCand) {
    const uint32_t rpi = item_rpi(W), q = r / rpi, it = st.g_item0[A] + q;
    *first_item = it;
    *n_start = (r == q * rpi) ? 1u : 0u;
    return it * (uint32_t)kItemCand + (r - q * rpi) * W;
  }
  const uint32_t nct = item_nct(W), it = st.g_item0[A] + r * nct;
  *first_item = it;
  *n_start = nct;
  return it * (uint32_t)kItemCand;
}
// count word of edge k (1 <= k <= 14): cum(k) = cum[k - 1] sits in u16 slot k - 1 of the 7 words q2.y .. q3.w
__device__ __forceinline__ uint32_t bin_cum(const uint4 &q2, const uint4 &q3, int k, uint32_t n) {
  if (k <= 0) return 0u;
  if (k >= kModBins) return n;
  const int wi = (k - 1) >> 1;
  const uint32_t w = wi == 0 ? q2.y : (wi == 1 ? q2.z : (wi == 2 ? q2.w : (wi == 3 ? q3.x : (wi == 4 ? q3.y : (wi == 5 ? q3.z : q3.w)))));
  return (k & 1) ? (w & 0xFFFFu) : (w >> 16);
}
struct LsWarpSh {
  uint32_t q1[3 * 64];
  ClStage cl;
  uint32_t seg_md[32], seg_key[32], seg_f[32], seg_row[32];
  float4 r_pos[kLsGrab];             // the grabbed rows: anchor
  float4 r_aux[kLsGrab];             // phi, kappa_MD, sigma_kappa_MD, category (as float bits)
  uint32_t r_key[kLsGrab], r_e0[kLsGrab], r_pre[kLsGrab + 1];   // key_base, first map edge, prefix of the degrees
};

// Tier 2 on up to 32 queued tier-1 survivors (dense lanes): cut L3 in its square-root-only mode-R form
// for an outer MD in a barrel module, the full fp32 pre-filter for an outer MD in an endcap module;
// what passes goes to the stage's candidate list.
__device__ __forceinline__ void ls_stage2(const SlotDev &s, const Params &g, WarpQueue3 &Q1, ClBuf &cl) {
  uint32_t mi = 0, mo = 0, key = 0;
  bool keep = false;
  if (Q1.pop(&mi, &mo, &key)) {
    const float4 a = s.md_pos[mi], b = s.md_pos[mo];
    const float2 ka = s.md_kf[mi], kb = s.md_kf[mo];
    const int ci = (int)(s.md_mod[mi] & 3u), co = (int)(s.md_mod[mo] & 3u);
    if (co < 2) keep = ls_l3_modeR_f(g, a.x, a.y, a.w, ka.x, ka.y, g.f_sig_t[ci], ci >= 2, b.x, b.y, b.w, kb.x, kb.y, g.f_sig_t[co]);
    else keep = ls_pre_f(g, a.x, a.y, a.z, a.w, ka.x, ka.y, ci, b.x, b.y, b.z, b.w, kb.x, kb.y, co);
  }
  cl.push(s.hdr, s.st[S_LS], S_LS, keep, key, make_uint2(mi, mo));
}

__global__ void __launch_bounds__(kThreads, 8) k_ls_eval(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B,
                                                         const __grid_constant__ Params g, int use_windows) {
  __shared__ LsWarpSh sh_all[kThreads / 32];
  __shared__ float4 tab[4];                     // per category: sig_z, sig_r, sig_t
  pdl_enter();
  LST_SLOT(B);
  const StageBuf &st = s.st[S_LS];
  const uint32_t n_md = s.hdr->n_obj[0];
  const int tid = threadIdx.x, lane = tid & 31;
  LsWarpSh &sh = sh_all[tid >> 5];
  if (tid < 4) tab[tid] = make_float4(g.f_sig_z[tid], g.f_sig_r[tid], g.f_sig_t[tid], 0.0f);
  __syncthreads();
  WarpQueue3 Q1;
  Q1.init(sh.q1);
  ClBuf cl;
  cl.init(&sh.cl);
  const uint32_t le_mask = 0xFFFFFFFFu >> (31 - lane);
  unsigned long long n_eval = 0;
  const bool live_stage = s.hdr->n_items[S_LS] != 0;     // 0: nothing to do, or the work list overflowed
  for (;;) {
    uint32_t r0 = 0;
    if (lane == 0) r0 = atomicAdd(&s.hdr->next_unit[S_LS], (uint32_t)kLsGrab);
    r0 = __shfl_sync(0xffffffffu, r0, 0);
    if (r0 >= n_md || !live_stage) break;
    // ---- lanes 0 .. kLsGrab-1 set up one row each
    uint32_t deg = 0, clr_item = 0, clr_n = 0;
    if (lane < kLsGrab && r0 + lane < n_md) {
      const uint32_t i = r0 + lane;
      const uint32_t mc = s.md_mod[i], A = mc >> 2;
      const uint32_t W = st.gW[A];
      if (W) {
        const float2 kf = s.md_kf[i];
        const uint32_t r = i - s.md_mod_off[A];
        const uint32_t key_base = ls_key_base(st, A, r, W, &clr_item, &clr_n);
        const uint32_t e0 = geo.map_off[A];
        deg = geo.map_off[A + 1] - e0;
        sh.r_pos[lane] = s.md_pos[i];
        sh.r_aux[lane] = make_float4(s.md_phi[i], kf.x, kf.y, __uint_as_float(mc & 3u));
        sh.r_key[lane] = key_base;
        sh.r_e0[lane] = e0;
      }
    }
    uint32_t P;
    const uint32_t dpre = warp_excl_scan(deg, &P);
    if (lane <= kLsGrab) sh.r_pre[lane] = dpre;             // r_pre[kLsGrab] = P (lanes >= kLsGrab have deg 0)
    // the row that starts a work item clears the item's pass bits (the decide kernel ORs them in)
#pragma unroll
    for (int q = 0; q < kLsGrab; ++q) {
      const uint32_t ci = __shfl_sync(0xffffffffu, clr_item, q), cn = __shfl_sync(0xffffffffu, clr_n, q);
      for (uint32_t w = lane; w < cn * (uint32_t)kItemWords; w += 32) st.mask[(size_t)ci * kItemWords + w] = 0;
    }
    __syncwarp();
    for (uint32_t pb = 0; pb < P; pb += 32) {
      // ---- lanes = (row, connected module) pairs: the range of the module's MDs the row has to look at
      const uint32_t pidx = pb + lane;
      uint32_t md0 = 0, len = 0, cB = 0, kcol = 0, k = 0;
      if (pidx < P) {
#pragma unroll
        for (int q = 1; q < kLsGrab; ++q) k += (sh.r_pre[q] <= pidx);
        const uint32_t e = sh.r_e0[k] + (pidx - sh.r_pre[k]);
        const uint4 *rec = reinterpret_cast<const uint4 *>(&s.mod_ev[geo.map_cols[e]]);
        const uint4 q2 = rec[2];
        const uint32_t n = q2.x & 0x3FFFFFFFu;
        if (n) {
          const uint4 q0 = rec[0], q1 = rec[1], q3 = rec[3];
          cB = q2.x >> 30;
          uint32_t lo = 0;
          len = n;
          if (use_windows) {
            const float4 a = sh.r_pos[k], ax = sh.r_aux[k];
            float w;
            if (!ls_row_window(g, a.w, a.z, (int)__float_as_uint(ax.w), __uint_as_float(q0.x), __uint_as_float(q0.y),
                               __uint_as_float(q0.z), __uint_as_float(q0.w), (int)cB, &w)) len = 0;
            else {
              const float pmin = __uint_as_float(q1.x), inv_w = __uint_as_float(q1.y);
              const float d = ax.x - __uint_as_float(q1.z);
              const float c = d - 6.2831853071795864769f * rintf(d * 0.15915494309189533577f);
              if (fabsf(c) + w < 3.0f && inv_w > 0.0f) {
                // no wrap-around inside [c - w, c + w]: the MDs whose key lies in it are a range; its ends
                // are rounded outwards to the bin edges (1e-5 rad covers the rounding of the edge positions)
                const float t_lo = (c - w - 1e-5f - pmin) * inv_w, t_hi = (c + w + 1e-5f - pmin) * inv_w;
                const int k_lo = t_lo >= (float)kModBins ? kModBins : (t_lo > 0.0f ? (int)t_lo : 0);
                const int k_hi = t_hi >= (float)(kModBins - 1) ? kModBins : (t_hi >= 0.0f ? (int)t_hi + 1 : 0);
                lo = bin_cum(q2, q3, k_lo, n);
                const uint32_t hi = bin_cum(q2, q3, k_hi, n);
                len = hi > lo ? hi - lo : 0u;
              }
            }
          }
          md0 = q1.w + lo;
          kcol = sh.r_key[k] + s.edge_col0[e] + lo;
        }
      }
      uint32_t T;
      const uint32_t fex = warp_excl_scan(len, &T);           // flat offset of the segment's first candidate
      const uint32_t bal = __ballot_sync(0xffffffffu, len != 0);
      const uint32_t nseg = __popc(bal);
      if (len) {
        const uint32_t pseg = __popc(bal & ((1u << lane) - 1u));
        sh.seg_md[pseg] = md0 | (cB << 30);
        sh.seg_key[pseg] = kcol;
        sh.seg_f[pseg] = fex;
        sh.seg_row[pseg] = k;
      }
      __syncwarp();
      n_eval += T;
      // ---- lanes = candidates of the concatenated ranges
      uint32_t sbefore = 0;                   // segments that start before the current 32 candidates
      for (uint32_t w0 = 0; w0 < T; w0 += 32) {
        const uint32_t sidx = sbefore + lane;
        uint32_t bit = 0;
        if (sidx < nseg) { const uint32_t f = sh.seg_f[sidx]; if (f < w0 + 32u) bit = 1u << (f - w0); }
        const uint32_t starts = __reduce_or_sync(0xffffffffu, bit);
        const uint32_t f = w0 + lane;
        bool keep = false;
        uint32_t mi = 0, mo = 0, key = 0;
        if (f < T) {
          const uint32_t sg = sbefore + __popc(starts & le_mask) - 1u;
          const uint32_t smd = sh.seg_md[sg], off = f - sh.seg_f[sg], kr = sh.seg_row[sg];
          mo = (smd & 0x3FFFFFFFu) + off;
          mi = r0 + kr;
          key = sh.seg_key[sg] + off;
          const float4 a = sh.r_pos[kr], ax = sh.r_aux[kr];
          const float4 b = s.md_pos[mo];
          const uint32_t ci = __float_as_uint(ax.w), co = smd >> 30;
          const float4 ta = tab[ci], tb = tab[co];
          keep = ls_tier1_f(g, a.x, a.y, a.z, a.w, ta.x, ta.y, ta.z, b.x, b.y, b.z, b.w, tb.x, tb.y, tb.z, co >= 2u);
        }
        sbefore += __popc(starts);
        Q1.push(keep, mi, mo, key);
        if (Q1.n >= 32u) ls_stage2(s, g, Q1, cl);
      }
      __syncwarp();                           // the segment table is rewritten by the next 32 pairs
    }
    __syncwarp();                             // ... and the row table by the next grab
  }
  while (Q1.n) ls_stage2(s, g, Q1, cl);
  cl.flush_all(s.hdr, st, S_LS);
  if (lane == 0 && n_eval) atomicAdd(&s.hdr->cand_eval[S_LS], n_eval);     // n_eval is warp-uniform
}

// fp64 decision of the listed candidates, one thread each (dense warps, no staging); an accepted
// candidate sets its pass bit and writes its results to the pool.
__global__ void __launch_bounds__(128) k_ls_decide(const __grid_constant__ Batch B, const __grid_constant__ Params g) {
  pdl_enter();
  LST_SLOT(B);
  const StageBuf &st = s.st[S_LS];
  Header *hdr = s.hdr;
  const uint32_t n = min(hdr->cl_used[S_LS], st.cap_cl);
  const uint32_t nround = (n + 31u) & ~31u;
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < nround; j += gridDim.x * blockDim.x) {
    bool pass = false;
    LsOut o;
    uint32_t key = 0;
    uint2 ab = make_uint2(0u, 0u);
    if (j < n) {
      key = st.cl_key[j]; ab = st.cl_ab[j];
      const float4 a = s.md_pos[ab.x], b = s.md_pos[ab.y];
      const double2 ka = s.md_kd[ab.x], kb = s.md_kd[ab.y];
      const Pt pa = make_pt(a.x, a.y, a.z, (int)(s.md_mod[ab.x] & 3u)), pb = make_pt(b.x, b.y, b.z, (int)(s.md_mod[ab.y] & 3u));
      pass = ls_eval_d(g, pa, ka.x, ka.y, pb, kb.x, kb.y, &o);
    }
    if (pass) {
      atomicOr(&st.mask[(size_t)(key / kItemCand) * kItemWords + ((key % kItemCand) >> 5)], 1u << (key & 31u));
      st.p_f4[j] = make_float4((float)o.dphi, (float)o.kappa, (float)o.sigk, 0.0f);
    }
  }
}

// One thread per pool entry: move it to its canonical position.  Then the LS range of every inner MD
// (ls_md_off) from the rank of the row's first candidate.
__global__ void __launch_bounds__(256) k_ls_fill(const __grid_constant__ Batch B) {
  pdl_enter();
  LST_SLOT(B);
  const StageBuf &st = s.st[S_LS];
  const Header *hdr = s.hdr;
  const uint32_t n_md = hdr->n_obj[0], n_ls = hdr->n_obj[1], n_items = hdr->n_items[S_LS];
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nt = gridDim.x * blockDim.x;
  for (uint32_t i = tid; i <= n_md; i += nt) {
    uint32_t off = n_ls;
    if (i < n_md) {
      const uint32_t A = s.md_mod[i] >> 2, W = st.gW[A];
      uint32_t key = st.g_item0[A] * (uint32_t)kItemCand, fi, ns;
      if (W) key = ls_key_base(st, A, i - s.md_mod_off[A], W, &fi, &ns);
      off = rank_before(st, n_items, n_ls, key);
    }
    s.ls_md_off[i] = off;
  }
  const uint32_t n = n_ls ? min(hdr->cl_used[S_LS], st.cap_cl) : 0u;
  for (uint32_t j = tid; j < n; j += nt) {
    const uint32_t idx = pool_target(st, st.cl_key[j]);
    if (idx == 0xFFFFFFFFu) continue;
    s.ls_md[idx] = st.cl_ab[j];
    st_f4(s, s.ls_f, idx, st.p_f4[j]);
  }
}

// ------------------------------------------------------------------ launchers
static inline int persistent_grid(const Ctx &c, int per_sm) { return c.n_sm * per_sm; }

void launch_md(const Ctx &c, const Batch &b, cudaStream_t st) {
  launch_k(c, st, "k_md_eval", k_md_eval, dim3(grid_for(b.s[0].cap_hits, 256, c.n_sm * 8)), 256, 0, false, c.geo, b, c.par);
  launch_k(c, st, "k_md_decide", k_md_decide, dim3(persistent_grid(c, 4)), 128, 0, false, c.geo, b, c.par);
  launch_counts(c, b, S_MD, 0, b.s[0].cap_md, false, st);
  launch_k(c, st, "k_md_fill", k_md_fill, dim3(persistent_grid(c, 4)), 256, 0, false, c.geo, b);
}

void launch_ls(const Ctx &c, const Batch &b, cudaStream_t st) {
  launch_k(c, st, "k_ls_groups", k_ls_groups, dim3((c.geo.n_modules + kLsGroupWarps - 1) / kLsGroupWarps), 32 * kLsGroupWarps, 0,
           false, c.geo, b);
  launch_k(c, st, "k_ls_eval", k_ls_eval, dim3(persistent_grid(c, 8)), kThreads, 0, false, c.geo, b, c.par, c.ls_windows);
  launch_k(c, st, "k_ls_decide", k_ls_decide, dim3(persistent_grid(c, 4)), 128, 0, false, b, c.par);
  launch_counts(c, b, S_LS, 1, b.s[0].cap_ls, false, st);
  launch_k(c, st, "k_ls_fill", k_ls_fill, dim3(persistent_grid(c, 4)), 256, 0, false, b);
}

}  // namespace lst
