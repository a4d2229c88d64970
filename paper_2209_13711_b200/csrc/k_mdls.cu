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

__global__ void __launch_bounds__(kThreads) k_ls_eval(GeoDev geo, SlotDev s, Params g) {
  __shared__ ItemScratch sc;
  __shared__ MapRow mr;
  __shared__ float4 p_pos[kItemCand + 8];
  __shared__ float2 p_kf[kItemCand + 8];
  __shared__ uint32_t p_idx[kItemCand + 8];
  __shared__ uint8_t p_cat[kItemCand + 8];
  const StageBuf &st = s.st[S_LS];
  const uint32_t n_items = s.hdr->n_items[S_LS];
  const int tid = threadIdx.x;
  for (uint32_t it = blockIdx.x; it < n_items; it += gridDim.x) {
    const Item item = st.items[it];
    const uint32_t A = item.group;
    const int nr = item.nrows, nj = item.nj;
    const uint32_t i0 = s.md_mod_off[A] + item.i0;
    stage_map_row(mr, geo, s, A);
    if (tid < kItemWords) sc.mask[tid] = 0;
    if (tid == 0) sc.n = 0;
    __syncthreads();
    for (int k = tid; k < nr + nj; k += kThreads) {
      const uint32_t md = k < nr ? i0 + k : map_col_to_md(mr, item.j0 + (k - nr));
      p_idx[k] = md;
      p_pos[k] = s.md_pos[md];
      p_kf[k] = s.md_kf[md];
      p_cat[k] = (uint8_t)(s.md_mod[md] & 3u);
    }
    __syncthreads();
    const int nc = nr * nj;
    for (int base = 0; base < nc; base += kThreads) {
      const int c = base + tid;
      bool keep = false;
      if (c < nc) {
        const int r = c / nj, jj = nr + (c - r * nj);
        const float4 a = p_pos[r], b = p_pos[jj];
        const float2 ka = p_kf[r], kb = p_kf[jj];
        keep = ls_pre_f(g, a.x, a.y, a.z, a.w, ka.x, ka.y, p_cat[r], b.x, b.y, b.z, b.w, kb.x, kb.y, p_cat[jj]);
      }
      push_survivor(sc, keep, (uint32_t)c);
    }
    __syncthreads();
    const int nsv = (int)sc.n;
    for (int k = tid; k < nsv; k += kThreads) {
      const int c = sc.list[k];
      const int r = c / nj, jj = nr + (c - r * nj);
      const float4 a = p_pos[r], b = p_pos[jj];
      const double2 ka = s.md_kd[p_idx[r]], kb = s.md_kd[p_idx[jj]];
      const Pt pa = make_pt(a.x, a.y, a.z, p_cat[r]), pb = make_pt(b.x, b.y, b.z, p_cat[jj]);
      if (ls_eval_d(g, pa, ka.x, ka.y, pb, kb.x, kb.y, nullptr)) atomicOr(&sc.mask[c >> 5], 1u << (c & 31));
    }
    __syncthreads();
    publish_mask(sc, st.mask + (size_t)it * kItemWords, st.item_cnt + it);
    __syncthreads();
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
  k_ls_eval<<<persistent_grid(c, 5), kThreads, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, "k_ls_eval");
  launch_scan_items(c, s, S_LS, 1, s.cap_ls, st);
  k_ls_fill<<<persistent_grid(c, 8), kThreads, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, "k_ls_fill");
  launch_row_offsets(c, s, 1, st);
}

}  // namespace lst
