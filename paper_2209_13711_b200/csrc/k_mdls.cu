// k_mdls.cu -- a1 mini-doublets (Fig. 2; reading C1) and a2 line segments
// (Fig. 4-7; reading C3).
#include "lst_launch.h"

namespace lst {

// =================================================================== MD
// Work item = (module, rows of lower hits, columns of upper hits), <= 1024 pairs (typically ~100).
// k_md_eval: one WARP per item, no staging and no barriers: every (lower, upper) pair goes through
// the fp32 pre-filter, the survivors are appended to the stage's candidate list.
// k_md_decide: one thread per listed pair, fp64 decision; accepted pairs set their pass bit and
// write kappa, sigma_kappa and dphi to the pool.
__global__ void __launch_bounds__(256) k_md_eval(GeoDev geo, SlotDev s, Params g) {
  __shared__ ClStageT<64> cl_mem[256 / 32];
  const StageBuf &st = s.st[S_MD];
  const uint32_t n_items = s.hdr->n_items[S_MD];
  const int lane = threadIdx.x & 31;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
  ClBufT<64> cl;
  cl.init(&cl_mem[threadIdx.x >> 5]);
  constexpr int kSlices = 8, kSliceCand = kItemCand / kSlices;   // a warp task = 128 candidates of an item
  for (uint32_t w = warp; w < n_items * kSlices; w += nwarp) {
    const uint32_t it = w / kSlices, sl = w % kSlices;
    const Item item = st.items[it];
    const int nj = item.nj, nc = item.nrows * nj;
    if (sl == 0) st.mask[(size_t)it * kItemWords + lane] = 0;  // the decide kernel ORs the pass bits in
    if ((int)(sl * kSliceCand) >= nc) continue;
    const uint32_t m = item.group;
    const int cat = geo.category[m];
    const uint32_t lo0 = s.det_off[2 * m] + item.i0, up0 = s.det_off[2 * m + 1] + item.j0;
    const uint32_t inv = (1u << 20) / (uint32_t)nj + 1u;      // c / nj == (c * inv) >> 20 for c * nj < 2^20
    const int c_end = min(nc, (int)((sl + 1) * kSliceCand));
    for (int base = (int)(sl * kSliceCand); base < c_end; base += 32) {
      const int c = base + lane;
      bool keep = false;
      uint32_t hl = 0, hu = 0;
      if (c < c_end) {
        const int r = (int)(((uint32_t)c * inv) >> 20), jj = c - r * nj;
        hl = lo0 + r; hu = up0 + jj;
        const float4 l = s.hit[hl], u = s.hit[hu];
        keep = md_pre_f(g, l.x, l.y, l.z, l.w, u.x, u.y, u.z, u.w, cat);
      }
      cl.push(s.hdr, st, S_MD, keep, it * (uint32_t)kItemCand + (uint32_t)c, make_uint2(hl, hu));
    }
  }
  cl.flush_all(s.hdr, st, S_MD);
}

__global__ void __launch_bounds__(128) k_md_decide(GeoDev geo, SlotDev s, Params g) {
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
      const int cat = geo.category[st.items[key / kItemCand].group];
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

// One thread per listed pair: the accepted ones move to their canonical position.
__global__ void __launch_bounds__(256) k_md_fill(GeoDev geo, SlotDev s) {
  const StageBuf &st = s.st[S_MD];
  const Header *hdr = s.hdr;
  if (hdr->n_obj[0] == 0) return;                            // nothing built, or overflow (level emptied)
  const uint32_t n = min(hdr->cl_used[S_MD], st.cap_cl);
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
    const uint32_t key = st.cl_key[j];
    const uint32_t idx = pool_target(st, key);
    if (idx == 0xFFFFFFFFu) continue;
    const uint32_t m = st.items[key / kItemCand].group;
    const uint2 h = st.cl_ab[j];
    const float4 l = s.hit[h.x];
    const double2 kd = st.p_d2[j];
    s.md_pos[idx] = l;
    s.md_kd[idx] = kd;
    s.md_kf[idx] = make_float2((float)kd.x, (float)kd.y);
    s.md_hit[idx] = h;
    s.md_mod[idx] = (m << 2) | (uint32_t)geo.category[m];
    s.md_dphi[idx] = st.p_f4[j].x;
    s.md_phi[idx] = atan2f(l.y, l.x);
    s.md_prel[idx] = s.hit_key[h.x];
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

// One block per WORK UNIT (k_emit_items): up to kUnitItems items of module A that share one column
// tile; the MDs of the connected modules (columns) and the unit's rows are staged in shared memory
// once (an inner-barrel module compares each of its ~30 MDs with ~1200 MDs of ~64 neighbours).
// After the staging the warps work independently, without block barriers: a warp owns 32 columns
// (kept in registers) and walks the rows (broadcast reads); three stages connected by warp queues:
//   tier 1 (ls_tier1_f: no division / sqrt / atan, ~82 % rejected) on every candidate,
//   tier 2 (ls_pre_f, full fp32) on 32 queued survivors at a time,
//   the fp64 decision on 32 queued tier-2 survivors at a time (~3 % of the candidates).
struct LsWarpMem {                    // the warps' queues: live only in the candidate phase of a unit
  uint32_t q1[kThreads / 32][64];
  ClStage cl[kThreads / 32];
};
struct LsShared {
  union {                             // the map row is needed only while the columns are staged
    MapRow mr;
    LsWarpMem w;
  };
  float4 c_pos[kItemCand];
  uint32_t c_idc[kItemCand];          // MD index | category << 30
  float4 r_pos[kUnitRows];
  uint32_t r_idc[kUnitRows];
  float4 tab[4];                      // per category: sig_z, sig_r, sig_t
};

// Tier 2 on up to 32 queued tier-1 survivors; what passes goes to the stage's candidate list.
// it0: item of the unit's first row chunk; consecutive row chunks are nct items apart.
__device__ __forceinline__ void ls_stage2(const LsShared &sh, const SlotDev &s, const Params &g, WarpQueue &Q1,
                                          ClBuf &cl, uint32_t rpi, int nj, uint32_t it0, uint32_t nct) {
  uint32_t e = 0, mi = 0, mo = 0, key = 0;
  bool keep = false;
  if (Q1.pop(&e)) {
    const uint32_t r = e & 0xFFu, jj = e >> 8;
    const float4 a = sh.r_pos[r], b = sh.c_pos[jj];
    const uint32_t ia = sh.r_idc[r], ib = sh.c_idc[jj];
    mi = ia & 0x3FFFFFFFu; mo = ib & 0x3FFFFFFFu;
    const float2 ka = s.md_kf[mi], kb = s.md_kf[mo];
    keep = ls_pre_f(g, a.x, a.y, a.z, a.w, ka.x, ka.y, (int)(ia >> 30), b.x, b.y, b.z, b.w, kb.x, kb.y, (int)(ib >> 30));
    const uint32_t q = r / rpi, c = (r - q * rpi) * (uint32_t)nj + jj;
    key = (it0 + q * nct) * (uint32_t)kItemCand + c;
  }
  cl.push(s.hdr, s.st[S_LS], S_LS, keep, key, make_uint2(mi, mo));
}

__global__ void __launch_bounds__(kThreads, 8) k_ls_eval(GeoDev geo, SlotDev s, Params g) {
  __shared__ LsShared sh;
  const StageBuf &st = s.st[S_LS];
  const uint32_t n_units = s.hdr->n_units[S_LS];
  const int tid = threadIdx.x, lane = tid & 31, wib = tid >> 5;
  constexpr int kWarps = kThreads / 32;
  if (tid < 4) sh.tab[tid] = make_float4(g.f_sig_z[tid], g.f_sig_r[tid], g.f_sig_t[tid], 0.0f);
  WarpQueue Q1;
  Q1.init(sh.w.q1[wib]);
  ClBuf cl;
  cl.init(&sh.w.cl[wib]);
  __shared__ uint32_t sh_unit[2];
  __shared__ int sh_task;                       // next (chunk, row group) task of the unit: warps take them dynamically
  for (;;) {
    __syncthreads();                            // the previous unit is done with the shared arrays
    if (tid == 0) {                             // units are handed out dynamically (their cost varies 100x)
      const uint32_t nu = atomicAdd(&s.hdr->next_unit[S_LS], 1u);
      sh_unit[0] = nu;
      sh_unit[1] = nu < n_units ? st.unit_group[nu] : 0u;
      sh_task = 0;
    }
    __syncthreads();
    const uint32_t u = sh_unit[0];
    if (u >= n_units) break;
    const uint32_t A = sh_unit[1], lu = u - st.g_unit0[A];
    const uint32_t R = st.gR[A], W = st.gW[A];
    const uint32_t nct = item_nct(W), rpi = item_rpi(W), ipu = unit_items(W);
    const uint32_t nq = (R + rpi - 1) / rpi;
    const uint32_t ct = lu % nct, q0 = (lu / nct) * ipu;
    const uint32_t qn = min(ipu, nq - q0);
    const uint32_t j0 = ct * kItemCand;
    const int nj = (int)min((uint32_t)kItemCand, W - j0);
    const uint32_t md0 = s.md_mod_off[A], item0 = st.g_item0[A];
    const uint32_t row0 = q0 * rpi, it0 = item0 + q0 * nct + ct;
    const int nrows = (int)min(R - row0, qn * rpi);      // <= kUnitRows
    stage_map_row(sh.mr, geo, s, A);
    for (int k = tid; k < nrows; k += kThreads) {
      const uint32_t md = md0 + row0 + k;
      sh.r_pos[k] = s.md_pos[md];
      sh.r_idc[k] = md | ((s.md_mod[md] & 3u) << 30);
    }
    for (int k = tid; k < (int)(qn * kItemWords); k += kThreads)      // the decide kernel ORs the pass bits in
      st.mask[(size_t)(it0 + (k / kItemWords) * nct) * kItemWords + (k % kItemWords)] = 0;
    __syncthreads();
    for (int k = tid; k < nj; k += kThreads) {
      const uint32_t md = map_col_to_md(sh.mr, j0 + k);
      sh.c_pos[k] = s.md_pos[md];
      sh.c_idc[k] = md | ((s.md_mod[md] & 3u) << 30);
    }
    __syncthreads();
    // tasks: (32-column chunk, interleaved row group); with few chunks the rows are split over the warps
    const int nchunk = (nj + 31) >> 5;
    const int nrg = nchunk >= kWarps ? 1 : kWarps / nchunk;
    for (;;) {
      int t = 0;
      if (lane == 0) t = atomicAdd(&sh_task, 1);
      t = __shfl_sync(0xffffffffu, t, 0);
      if (t >= nchunk * nrg) break;
      const int chunk = t % nchunk, rg = t / nchunk;
      const int jj = chunk * 32 + lane;
      const bool has = jj < nj;
      const float4 b = sh.c_pos[has ? jj : 0];
      const uint32_t cb = sh.c_idc[has ? jj : 0] >> 30;
      const float4 tb = sh.tab[cb];
      // the 32 columns of a chunk nearly always share their mode (same or neighbouring modules):
      // a warp-uniform mode lets the compiler drop the other mode's arithmetic from the loop
      const bool all_z = __all_sync(0xffffffffu, !has || cb >= 2u), all_r = __all_sync(0xffffffffu, !has || cb < 2u);
#define LST_LS_ROWS(OEC)                                                                                             \
      for (int r = rg; r < nrows; r += nrg) {                                                                        \
        const float4 a = sh.r_pos[r];                                                                                \
        const float4 ta = sh.tab[sh.r_idc[r] >> 30];                                                                 \
        const bool keep = has && ls_tier1_f(g, a.x, a.y, a.z, a.w, ta.x, ta.y, ta.z, b.x, b.y, b.z, b.w, tb.x, tb.y, \
                                            tb.z, (OEC));                                                            \
        Q1.push(keep, (uint32_t)r | ((uint32_t)jj << 8));                                                            \
        if (Q1.n >= 32u) ls_stage2(sh, s, g, Q1, cl, rpi, nj, it0, nct);                                             \
      }
      if (all_r) { LST_LS_ROWS(false) }
      else if (all_z) { LST_LS_ROWS(true) }
      else { LST_LS_ROWS(cb >= 2u) }
#undef LST_LS_ROWS
    }
    while (Q1.n) ls_stage2(sh, s, g, Q1, cl, rpi, nj, it0, nct);
    cl.flush_all(s.hdr, st, S_LS);      // the queues' memory is the next unit's map row
  }
}

// fp64 decision of the listed candidates, one thread each (dense warps, no staging); an accepted
// candidate sets its pass bit and writes its results to the pool.
__global__ void __launch_bounds__(128) k_ls_decide(SlotDev s, Params g) {
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

// One thread per pool entry: move it to its canonical position.
__global__ void __launch_bounds__(256) k_ls_fill(SlotDev s) {
  const StageBuf &st = s.st[S_LS];
  const Header *hdr = s.hdr;
  if (hdr->n_obj[1] == 0) return;
  const uint32_t n = min(hdr->cl_used[S_LS], st.cap_cl);
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
    const uint32_t idx = pool_target(st, st.cl_key[j]);
    if (idx == 0xFFFFFFFFu) continue;
    s.ls_md[idx] = st.cl_ab[j];
    s.ls_f[idx] = st.p_f4[j];
  }
}

// ------------------------------------------------------------------ launchers
static inline int persistent_grid(const Ctx &c, int per_sm) { return c.n_sm * per_sm; }

void launch_md(const Ctx &c, const SlotDev &s, cudaStream_t st) {
  launch_emit(c, s, S_MD, -1, st);
  k_md_eval<<<persistent_grid(c, 8), 256, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, "k_md_eval");
  k_md_decide<<<persistent_grid(c, 4), 128, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, "k_md_decide");
  launch_item_counts(c, s, S_MD, st);
  launch_scan_items(c, s, S_MD, 0, s.cap_md, st);
  k_md_fill<<<persistent_grid(c, 4), 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_md_fill");
  launch_row_offsets(c, s, 0, st);
}

void launch_ls(const Ctx &c, const SlotDev &s, cudaStream_t st) {
  k_ls_groups<<<(c.geo.n_modules + 127) / 128, 128, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_ls_groups");
  launch_emit(c, s, S_LS, -1, st);
  k_ls_eval<<<persistent_grid(c, 8), kThreads, 0, st>>>(c.geo, s, c.par); LST_MARK(c, st, "k_ls_eval");
  k_ls_decide<<<persistent_grid(c, 4), 128, 0, st>>>(s, c.par); LST_MARK(c, st, "k_ls_decide");
  launch_item_counts(c, s, S_LS, st);
  launch_scan_items(c, s, S_LS, 1, s.cap_ls, st);
  k_ls_fill<<<persistent_grid(c, 4), 256, 0, st>>>(s); LST_MARK(c, st, "k_ls_fill");
  launch_row_offsets(c, s, 1, st);
}

}  // namespace lst
