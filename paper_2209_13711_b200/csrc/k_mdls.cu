// k_mdls.cu -- a1 mini-doublets (Fig. 2; reading C1) and a2 line segments
// (Fig. 4-7; reading C3).
#include "lst_launch.h"

namespace lst {

// =================================================================== MD
// Work item = (module, rows of lower hits, columns of upper hits).  Both sensors' hits are staged in
// shared memory; every (lower, upper) pair goes through the fp32 pre-filter, survivors are compacted
// and decided in fp64.
__global__ void __launch_bounds__(kThreads) k_md_eval(GeoDev geo, SlotDev s, Params g) {
  __shared__ ItemScratch sc;
  __shared__ float4 pool[kItemCand + 8];
  const StageBuf &st = s.st[S_MD];
  const uint32_t n_items = s.hdr->n_items[S_MD];
  const int tid = threadIdx.x;
  for (uint32_t it = blockIdx.x; it < n_items; it += gridDim.x) {
    const Item item = st.items[it];
    const uint32_t m = item.group;
    const int cat = geo.category[m];
    const uint32_t lo0 = s.det_off[2 * m] + item.i0, up0 = s.det_off[2 * m + 1] + item.j0;
    const int nr = item.nrows, nj = item.nj;
    for (int k = tid; k < nr + nj; k += kThreads) pool[k] = k < nr ? s.hit[lo0 + k] : s.hit[up0 + (k - nr)];
    if (tid < kItemWords) sc.mask[tid] = 0;
    if (tid == 0) sc.n = 0;
    __syncthreads();
    const int nc = nr * nj;
    for (int base = 0; base < nc; base += kThreads) {
      const int c = base + tid;
      bool keep = false;
      if (c < nc) {
        const int r = c / nj, jj = c - r * nj;
        const float4 l = pool[r], u = pool[nr + jj];
        keep = md_pre_f(g, l.x, l.y, l.z, l.w, u.x, u.y, u.z, u.w, cat);
      }
      push_survivor(sc, keep, (uint32_t)c);
    }
    __syncthreads();
    const int nsv = (int)sc.n;
    for (int k = tid; k < nsv; k += kThreads) {
      const int c = sc.list[k];
      const int r = c / nj, jj = c - r * nj;
      const float4 l = pool[r], u = pool[nr + jj];
      const Pt pl = make_pt(l.x, l.y, l.z, cat), pu = make_pt(u.x, u.y, u.z, cat);
      if (md_eval_d(g, pl, pu, cat, nullptr)) atomicOr(&sc.mask[c >> 5], 1u << (c & 31));
    }
    __syncthreads();
    publish_mask(sc, st.mask + (size_t)it * kItemWords, st.item_cnt + it);
    __syncthreads();
  }
}

__global__ void __launch_bounds__(kThreads) k_md_fill(GeoDev geo, SlotDev s, Params g) {
  __shared__ ItemScratch sc;
  const StageBuf &st = s.st[S_MD];
  const uint32_t n_items = s.hdr->n_items[S_MD];
  const int tid = threadIdx.x;
  for (uint32_t it = blockIdx.x; it < n_items; it += gridDim.x) {
    if (st.item_cnt[it] == 0) continue;   // uniform per block
    const Item item = st.items[it];
    const uint32_t m = item.group;
    const int cat = geo.category[m];
    const uint32_t lo0 = s.det_off[2 * m] + item.i0, up0 = s.det_off[2 * m + 1] + item.j0;
    const int nj = item.nj;
    expand_mask(sc, st.mask + (size_t)it * kItemWords);
    const int n = (int)sc.n;
    const uint32_t base = st.item_base[it];
    for (int k = tid; k < n; k += kThreads) {
      const int c = sc.list[k];
      const int r = c / nj, jj = c - r * nj;
      const uint32_t hl = lo0 + r, hu = up0 + jj;
      const float4 l = s.hit[hl], u = s.hit[hu];
      const Pt pl = make_pt(l.x, l.y, l.z, cat), pu = make_pt(u.x, u.y, u.z, cat);
      MdOut o;
      md_eval_d(g, pl, pu, cat, &o);
      const uint32_t idx = base + k;
      s.md_pos[idx] = l;
      s.md_kd[idx] = make_double2(o.kappa, o.sigk);
      s.md_kf[idx] = make_float2((float)o.kappa, (float)o.sigk);
      s.md_hit[idx] = make_uint2(hl, hu);
      s.md_mod[idx] = (m << 2) | (uint32_t)cat;
      s.md_dphi[idx] = (float)o.dphi;
      s.md_phi[idx] = atan2f(l.y, l.x);
    }
    __syncthreads();
  }
}

// =================================================================== LS
// Group of module A: rows = MDs of A, width W_A = number of MDs in the modules connected to A.
__global__ void k_ls_groups(GeoDev geo, SlotDev s) {
  const StageBuf &st = s.st[S_LS];
  for (uint32_t A = blockIdx.x * blockDim.x + threadIdx.x; A < geo.n_modules; A += gridDim.x * blockDim.x) {
    const uint32_t R = s.md_mod_off[A + 1] - s.md_mod_off[A];
    uint32_t W = 0;
    if (R) {
      for (uint32_t e = geo.map_off[A]; e < geo.map_off[A + 1]; ++e) {
        const uint32_t B = geo.map_cols[e];
        W += s.md_mod_off[B + 1] - s.md_mod_off[B];
      }
    }
    st.gR[A] = R;
    st.gW[A] = W;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) s.hdr->n_groups[S_LS] = geo.n_modules;
}

// Stage the module-map row of A: per connected module its first MD and the running MD count.
struct MapRow {
  uint32_t start[kMaxDeg];
  uint32_t cum[kMaxDeg + 1];
  int deg;
};
__device__ __forceinline__ void stage_map_row(MapRow &mr, const GeoDev &geo, const SlotDev &s, uint32_t A) {
  const int tid = threadIdx.x;
  const uint32_t e0 = geo.map_off[A];
  const int deg = (int)(geo.map_off[A + 1] - e0);
  if (tid == 0) mr.deg = deg;
  // deg <= kMaxDeg: sequential warp scan over the row by warp 0
  if (tid < 32) {
    uint32_t carry = 0;
    for (int b = 0; b < deg; b += 32) {
      const int e = b + tid;
      uint32_t n = 0, st0 = 0;
      if (e < deg) {
        const uint32_t B = geo.map_cols[e0 + e];
        st0 = s.md_mod_off[B];
        n = s.md_mod_off[B + 1] - st0;
      }
      uint32_t tot;
      const uint32_t ex = warp_excl_scan(n, &tot);
      if (e < deg) { mr.start[e] = st0; mr.cum[e] = carry + ex; }
      carry += tot;
    }
    if (tid == 0) mr.cum[deg] = carry;
  }
}
// column j of A's candidate list -> MD index
__device__ __forceinline__ uint32_t map_col_to_md(const MapRow &mr, uint32_t j) {
  int lo = 0, hi = mr.deg;            // find last e with cum[e] <= j
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (mr.cum[mid] <= j) lo = mid; else hi = mid;
  }
  return mr.start[lo] + (j - mr.cum[lo]);
}

// append candidate c to a survivor list (warp-aggregated shared atomic); all 32 lanes must call
__device__ __forceinline__ void push_list(uint16_t *list, uint32_t *n, bool keep, uint32_t c) {
  const uint32_t b = __ballot_sync(0xffffffffu, keep);
  if (b == 0) return;
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(b) - 1;
  uint32_t base = 0;
  if (lane == leader) base = atomicAdd(n, (uint32_t)__popc(b));
  base = __shfl_sync(0xffffffffu, base, leader);
  if (keep) list[base + __popc(b & ((1u << lane) - 1u))] = (uint16_t)c;
}

// One block per WORK UNIT (k_emit_items): up to kUnitItems items of module A that share one column
// tile, i.e. the MDs of the connected modules are staged in shared memory once and re-used for all
// rows (an inner-barrel module compares each of its ~30 MDs with ~1200 MDs of ~64 neighbours).
// Per item: tier 1 (ls_tier1_f: no division / sqrt / atan, ~82 % rejected) on every candidate,
// tier 2 (ls_pre_f, full fp32) on the compacted survivors, fp64 decision on what is left (~3 %).
__global__ void __launch_bounds__(kThreads) k_ls_eval(GeoDev geo, SlotDev s, Params g) {
  __shared__ ItemScratch sc;
  __shared__ uint16_t list2[kItemCand];
  __shared__ uint32_t n2;
  __shared__ MapRow mr;
  __shared__ float4 p_pos[kItemCand + 8];
  __shared__ uint32_t p_idc[kItemCand + 8];     // MD index | category << 30
  __shared__ float4 tab[4];                     // per category: sig_z, sig_r, sig_t
  const StageBuf &st = s.st[S_LS];
  const uint32_t n_units = s.hdr->n_units[S_LS], ng = s.hdr->n_groups[S_LS];
  const int tid = threadIdx.x;
  if (tid < 4) tab[tid] = make_float4(g.f_sig_z[tid], g.f_sig_r[tid], g.f_sig_t[tid], 0.0f);
  for (uint32_t u = blockIdx.x; u < n_units; u += gridDim.x) {
    uint32_t lo = 0, hi = ng;                   // last group with g_unit0 <= u
    while (hi - lo > 1) {
      const uint32_t mid = (lo + hi) >> 1;
      if (st.g_unit0[mid] <= u) lo = mid; else hi = mid;
    }
    const uint32_t A = lo, lu = u - st.g_unit0[A];
    const uint32_t R = st.gR[A], W = st.gW[A];
    const uint32_t nct = W <= (uint32_t)kItemCand ? 1u : (W + kItemCand - 1) / kItemCand;
    const uint32_t rpi = W <= (uint32_t)kItemCand ? (uint32_t)kItemCand / W : 1u;
    const uint32_t nq = (R + rpi - 1) / rpi;
    const uint32_t ct = lu % nct, q0 = (lu / nct) * kUnitItems;
    const uint32_t qn = min((uint32_t)kUnitItems, nq - q0);
    const uint32_t j0 = ct * kItemCand;
    const int nj = (int)min((uint32_t)kItemCand, W - j0);
    const uint32_t md0 = s.md_mod_off[A], item0 = st.g_item0[A];
    __syncthreads();                            // the previous unit is done with mr / p_pos
    stage_map_row(mr, geo, s, A);
    __syncthreads();
    for (int k = tid; k < nj; k += kThreads) {
      const uint32_t md = map_col_to_md(mr, j0 + k);
      p_pos[k] = s.md_pos[md];
      p_idc[k] = md | ((s.md_mod[md] & 3u) << 30);
    }
    const uint32_t inv = (1u << 20) / (uint32_t)nj + 1u;   // c / nj == (c * inv) >> 20 for c * nj < 2^20
    for (uint32_t qi = 0; qi < qn; ++qi) {
      const uint32_t q = q0 + qi, it = item0 + q * nct + ct, i0 = q * rpi;
      const int nr = (int)min(rpi, R - i0);
      for (int k = tid; k < nr; k += kThreads) {
        const uint32_t md = md0 + i0 + k;
        p_pos[nj + k] = s.md_pos[md];
        p_idc[nj + k] = md | ((s.md_mod[md] & 3u) << 30);
      }
      if (tid < kItemWords) sc.mask[tid] = 0;
      if (tid == 0) { sc.n = 0; n2 = 0; }
      __syncthreads();
      const int nc = nr * nj;
      for (int base = 0; base < nc; base += kThreads) {          // tier 1
        const int c = base + tid;
        bool keep = false;
        if (c < nc) {
          const int r = (int)(((uint32_t)c * inv) >> 20), jj = c - r * nj;
          const float4 a = p_pos[nj + r], b = p_pos[jj];
          const uint32_t ca = p_idc[nj + r] >> 30, cb = p_idc[jj] >> 30;
          const float4 ta = tab[ca], tb = tab[cb];
          keep = ls_tier1_f(g, a.x, a.y, a.z, a.w, ta.x, ta.y, ta.z, b.x, b.y, b.z, b.w, tb.x, tb.y, tb.z, cb >= 2u);
        }
        push_list(sc.list, &sc.n, keep, (uint32_t)c);
      }
      __syncthreads();
      const int n1 = (int)sc.n;
      for (int base = 0; base < n1; base += kThreads) {          // tier 2
        const int k = base + tid;
        bool keep = false;
        int c = 0;
        if (k < n1) {
          c = sc.list[k];
          const int r = (int)(((uint32_t)c * inv) >> 20), jj = c - r * nj;
          const float4 a = p_pos[nj + r], b = p_pos[jj];
          const uint32_t ia = p_idc[nj + r], ib = p_idc[jj];
          const float2 ka = s.md_kf[ia & 0x3FFFFFFFu], kb = s.md_kf[ib & 0x3FFFFFFFu];
          keep = ls_pre_f(g, a.x, a.y, a.z, a.w, ka.x, ka.y, (int)(ia >> 30), b.x, b.y, b.z, b.w, kb.x, kb.y, (int)(ib >> 30));
        }
        push_list(list2, &n2, keep, (uint32_t)c);
      }
      __syncthreads();
      const int nsv = (int)n2;
      for (int k = tid; k < nsv; k += kThreads) {                // fp64 decision
        const int c = list2[k];
        const int r = (int)(((uint32_t)c * inv) >> 20), jj = c - r * nj;
        const float4 a = p_pos[nj + r], b = p_pos[jj];
        const uint32_t ia = p_idc[nj + r], ib = p_idc[jj];
        const double2 ka = s.md_kd[ia & 0x3FFFFFFFu], kb = s.md_kd[ib & 0x3FFFFFFFu];
        const Pt pa = make_pt(a.x, a.y, a.z, (int)(ia >> 30)), pb = make_pt(b.x, b.y, b.z, (int)(ib >> 30));
        if (ls_eval_d(g, pa, ka.x, ka.y, pb, kb.x, kb.y, nullptr)) atomicOr(&sc.mask[c >> 5], 1u << (c & 31));
      }
      __syncthreads();
      publish_mask(sc, st.mask + (size_t)it * kItemWords, st.item_cnt + it);
      __syncthreads();
    }
  }
}

__global__ void __launch_bounds__(kThreads) k_ls_fill(GeoDev geo, SlotDev s, Params g) {
  __shared__ ItemScratch sc;
  __shared__ MapRow mr;
  const StageBuf &st = s.st[S_LS];
  const uint32_t n_items = s.hdr->n_items[S_LS];
  const int tid = threadIdx.x;
  for (uint32_t it = blockIdx.x; it < n_items; it += gridDim.x) {
    if (st.item_cnt[it] == 0) continue;
    const Item item = st.items[it];
    const uint32_t A = item.group;
    const int nj = item.nj;
    const uint32_t i0 = s.md_mod_off[A] + item.i0;
    stage_map_row(mr, geo, s, A);
    expand_mask(sc, st.mask + (size_t)it * kItemWords);   // contains the __syncthreads the staging needs
    const int n = (int)sc.n;
    const uint32_t base = st.item_base[it];
    for (int k = tid; k < n; k += kThreads) {
      const int c = sc.list[k];
      const int r = c / nj, jj = c - r * nj;
      const uint32_t mi = i0 + r, mo = map_col_to_md(mr, item.j0 + jj);
      const float4 a = s.md_pos[mi], b = s.md_pos[mo];
      const double2 ka = s.md_kd[mi], kb = s.md_kd[mo];
      const Pt pa = make_pt(a.x, a.y, a.z, s.md_mod[mi] & 3u), pb = make_pt(b.x, b.y, b.z, s.md_mod[mo] & 3u);
      LsOut o;
      ls_eval_d(g, pa, ka.x, ka.y, pb, kb.x, kb.y, &o);
      const uint32_t idx = base + k;
      s.ls_md[idx] = make_uint2(mi, mo);
      s.ls_f[idx] = make_float4((float)o.dphi, (float)o.kappa, (float)o.sigk, 0.0f);
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------ launchers
static inline int persistent_grid(const Ctx &c, int per_sm) { return c.n_sm * per_sm; }

void launch_md(const Ctx &c, const SlotDev &s, cudaStream_t st) {
  launch_emit(c, s, S_MD, -1, st);
  k_md_eval<<<persistent_grid(c, 8), kThreads, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, "k_md_eval");
  launch_scan_items(c, s, S_MD, 0, s.cap_md, st);
  k_md_fill<<<persistent_grid(c, 8), kThreads, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, "k_md_fill");
  launch_row_offsets(c, s, 0, st);
}

void launch_ls(const Ctx &c, const SlotDev &s, cudaStream_t st) {
  k_ls_groups<<<(c.geo.n_modules + 127) / 128, 128, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_ls_groups");
  launch_emit(c, s, S_LS, -1, st);
  k_ls_eval<<<persistent_grid(c, 6), kThreads, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, "k_ls_eval");
  launch_scan_items(c, s, S_LS, 1, s.cap_ls, st);
  k_ls_fill<<<persistent_grid(c, 8), kThreads, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, "k_ls_fill");
  launch_row_offsets(c, s, 1, st);
}

}  // namespace lst
