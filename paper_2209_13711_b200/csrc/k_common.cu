// k_common.cu -- a0 hit indexing (PAPER.md:125 SoA event data) and the generic
// work-list kernels (emit items, scan item counts, row offsets) used by every stage.
#include "lst_launch.h"

namespace lst {

// ------------------------------------------------------------------ begin: reset the slot header
__global__ void k_begin(SlotDev s) {
  Header *h = s.hdr;
  const int t = threadIdx.x;
  if (t < 8) h->n_obj[t] = 0;
  if (t < S_NSTAGE) { h->n_items[t] = 0; h->n_groups[t] = 0; h->n_units[t] = 0; h->next_unit[t] = 0; h->cl_used[t] = 0; h->cand[t] = 0ull; h->cand_eval[t] = 0ull; }
  if (t == 0) { h->err = 0; h->n_inc = 0; h->n_heavy = 0; h->n_dd = 0; h->n_flag = 0; s.scan_part[kScanBlocks + 1] = 0; }
}

// ------------------------------------------------------------------ a0.1 histogram of det ids
__global__ void k_hist(GeoDev geo, SlotDev s) {
  const uint32_t n = s.hdr->n_hits;
  for (uint32_t h = blockIdx.x * blockDim.x + threadIdx.x; h < n; h += gridDim.x * blockDim.x) {
    const uint32_t d = s.raw_det[h];
    if (d >= geo.n_det) { atomicOr(&s.hdr->err, (uint32_t)ERR_DET); continue; }
    atomicAdd(&s.det_cnt[d], 1u);
    // input validation (include/lst.h): finite coordinates; a lower-sensor hit inside its module's box
    // (the dead-edge pruning of lst_create and the pixel-seed windows rely on the boxes)
    const float x = s.raw_x[h], y = s.raw_y[h], z = s.raw_z[h];
    if (!(fabsf(x) <= 3.0e38f && fabsf(y) <= 3.0e38f && fabsf(z) <= 3.0e38f)) { atomicOr(&s.hdr->err, (uint32_t)ERR_NONFINITE); continue; }
    if ((d & 1u) == 0u) {
      const uint32_t m = d >> 1;
      const float r = sqrtf(x * x + y * y);
      const float dp = atan2f(y, x) - geo.phic[m];
      const float dphi = fabsf(dp - 6.2831853071795864769f * rintf(dp * 0.15915494309189533577f));
      const bool in = r >= geo.rmin[m] - kBoxTolLen && r <= geo.rmax[m] + kBoxTolLen && z >= geo.zmin[m] - kBoxTolLen &&
                      z <= geo.zmax[m] + kBoxTolLen && dphi <= geo.hphi[m] + kBoxTolPhi + 4e-7f * (fabsf(geo.phic[m]) + 3.2f);
      if (!in) atomicOr(&s.hdr->err, (uint32_t)ERR_BOX);
    }
  }
}

// Exclusive scan of in[0..n) into out[0..n], out[n] = total; one block.
// Each thread owns a contiguous chunk (serial sum, ONE block scan of the chunk sums, serial write):
// two barriers in all instead of two per blockDim.x elements.  in == out is allowed.
__device__ void block_scan_array(const uint32_t *in, uint32_t *out, uint32_t n, uint32_t *sh) {
  const uint32_t chunk = (n + blockDim.x - 1) / blockDim.x;
  const uint32_t b0 = min(n, threadIdx.x * chunk), b1 = min(n, b0 + chunk);
  uint32_t sum = 0;
  for (uint32_t i = b0; i < b1; ++i) sum += in[i];
  uint32_t tot;
  uint32_t run = block_excl_scan(sum, sh, &tot);
  for (uint32_t i = b0; i < b1; ++i) { const uint32_t v = in[i]; out[i] = run; run += v; }
  if (threadIdx.x == 0) out[n] = tot;
}

// ------------------------------------------------------------------ a0.2 scan + MD groups
// det_off = exclusive scan of det_cnt; MD group of module m: rows = lower hits, width = upper hits.
__global__ void k_det_scan(GeoDev geo, SlotDev s) {
  __shared__ uint32_t sh[33];
  block_scan_array(s.det_cnt, s.det_off, geo.n_det, sh);
  __syncthreads();
  for (uint32_t d = threadIdx.x; d < geo.n_det; d += blockDim.x) s.det_cur[d] = 0;
  const StageBuf &st = s.st[S_MD];
  for (uint32_t m = threadIdx.x; m < geo.n_modules; m += blockDim.x) {
    st.gR[m] = s.det_cnt[2 * m];
    st.gW[m] = s.det_cnt[2 * m + 1];
  }
  if (threadIdx.x == 0) s.hdr->n_groups[S_MD] = geo.n_modules;
}

// ------------------------------------------------------------------ a0.3 scatter (unordered within a det)
__global__ void k_scatter(GeoDev geo, SlotDev s) {
  const uint32_t n = s.hdr->n_hits;
  for (uint32_t h = blockIdx.x * blockDim.x + threadIdx.x; h < n; h += gridDim.x * blockDim.x) {
    const uint32_t d = s.raw_det[h];
    if (d >= geo.n_det) continue;
    const uint32_t p = s.det_off[d] + atomicAdd(&s.det_cur[d], 1u);
    s.tmp_orig[p] = h;
    const float dphi = atan2f(s.raw_y[h], s.raw_x[h]) - geo.phic[d >> 1];
    const float key = dphi - 6.2831853071795864769f * rintf(dphi * 0.15915494309189533577f);
    s.tmp_key[p] = key == key ? key : 0.0f;      // NaN coordinates must not break the ranking
  }
}

// ------------------------------------------------------------------ a0.4 rank inside the det
// Makes the order canonical whatever order the atomics gave: inside a det the hits ascend in
// azimuth relative to the module centre (ties: caller index).  MDs (anchor = lower hit) and the
// T3 / T5 grouped by first MD are then azimuth-ordered inside a module, which the pixel joins use
// to cut a (seed, module) row down to the objects inside the seed's azimuthal window.
__global__ void k_rank(GeoDev geo, SlotDev s) {
  const uint32_t n = s.det_off[geo.n_det];
  for (uint32_t p = blockIdx.x * blockDim.x + threadIdx.x; p < n; p += gridDim.x * blockDim.x) {
    const uint32_t h = s.tmp_orig[p];
    const uint32_t d = s.raw_det[h];
    const uint32_t b = s.det_off[d], e = s.det_off[d + 1];
    const float key = s.tmp_key[p];
    uint32_t r = 0;
    for (uint32_t q = b; q < e; ++q) {
      const float kq = s.tmp_key[q];
      r += (kq < key || (kq == key && s.tmp_orig[q] < h));
    }
    const float x = s.raw_x[h], y = s.raw_y[h], z = s.raw_z[h];
    s.hit[b + r] = make_float4(x, y, z, sqrtf(x * x + y * y));
    s.hit_orig[b + r] = h;
    s.hit_key[b + r] = key;
  }
}

// ------------------------------------------------------------------ emit work items
__device__ __forceinline__ uint32_t items_of(uint32_t R, uint32_t W) {
  if (R == 0 || W == 0) return 0;
  const uint32_t rpi = item_rpi(W);
  return ((R + rpi - 1) / rpi) * item_nct(W);
}
// Work units of a group: the items (q, ct), q = row chunk, ct = column tile, are cut into runs of
// kUnitItems consecutive q at fixed ct; the items of a unit share their columns (item index of
// (q, ct) = g_item0 + q * n_ct + ct; unit u of the group: ct = u % n_ct, q0 = (u / n_ct) * unit_items(W)).
__device__ __forceinline__ uint32_t units_of(uint32_t R, uint32_t W) {
  if (R == 0 || W == 0) return 0;
  const uint32_t nct = item_nct(W), ipu = unit_items(W);
  const uint32_t nq = items_of(R, W) / nct;
  return nct * ((nq + ipu - 1) / ipu);
}

// One block.  rows_level >= 0: the groups are kRowChunk-row chunks of that object level and the
// kernel sets n_groups itself (gR must be 1, gW the group's candidate count: written by the
// stage's group kernel for every g < ceil(n_rows / kRowChunk)).
__global__ void k_emit_items(SlotDev s, int stage, int rows_level) {
  __shared__ uint32_t sh[33];
  __shared__ unsigned long long sh_cand;
  Header *hdr = s.hdr;
  const StageBuf &st = s.st[stage];
  uint32_t ng;
  if (rows_level >= 0) ng = (hdr->n_obj[rows_level] + kRowChunk - 1) / kRowChunk;
  else ng = hdr->n_groups[stage];
  if (ng > st.cap_groups) ng = 0;   // cannot happen: cap_groups is sized from the object capacity
  if (threadIdx.x == 0) sh_cand = 0ull;
  __syncthreads();
  // each thread owns a contiguous chunk of groups: serial sums, one block scan per quantity, serial write
  unsigned long long my_cand = 0;
  const uint32_t chunk = (ng + blockDim.x - 1) / blockDim.x;
  const uint32_t g0 = min(ng, threadIdx.x * chunk), g1 = min(ng, g0 + chunk);
  uint32_t si = 0, su = 0;
  for (uint32_t g = g0; g < g1; ++g) {
    const uint32_t R = st.gR[g], W = st.gW[g];
    si += items_of(R, W);
    su += units_of(R, W);
    my_cand += (unsigned long long)R * W;
  }
  uint32_t carry, ucarry;
  uint32_t ri = block_excl_scan(si, sh, &carry);
  __syncthreads();
  uint32_t ru = block_excl_scan(su, sh, &ucarry);
  for (uint32_t g = g0; g < g1; ++g) {
    const uint32_t R = st.gR[g], W = st.gW[g];
    st.g_item0[g] = ri; st.g_unit0[g] = ru;
    ri += items_of(R, W);
    ru += units_of(R, W);
  }
  // block sum of the candidate counts (64-bit shared atomics are CAS loops: reduce per warp first)
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) my_cand += __shfl_xor_sync(0xffffffffu, my_cand, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(&sh_cand, my_cand);
  __syncthreads();
  const bool overflow = carry > st.cap_items;
  if (threadIdx.x == 0) {
    st.g_item0[ng] = carry;
    st.g_unit0[ng] = ucarry;
    hdr->n_groups[stage] = ng;
    hdr->n_items[stage] = overflow ? 0u : carry;
    hdr->n_units[stage] = overflow ? 0u : ucarry;
    hdr->cand[stage] = sh_cand;
    if (overflow) atomicOr(&hdr->err, (uint32_t)ERR_CAP_ITEMS);
  }
}

// One thread per ITEM (a heavy module owns hundreds of items) and per UNIT: find its group in the
// offsets k_emit_items wrote; many blocks (the binary searches are latency bound).
__global__ void __launch_bounds__(256) k_emit_fill(SlotDev s, int stage) {
  const Header *hdr = s.hdr;
  const StageBuf &st = s.st[stage];
  const uint32_t ng = hdr->n_groups[stage], n_items = hdr->n_items[stage], n_units = hdr->n_units[stage];
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nt = gridDim.x * blockDim.x;
  for (uint32_t i = tid; i < n_items; i += nt) {
    uint32_t lo = 0, hi = ng;            // last g with g_item0[g] <= i (empty groups repeat an offset)
    while (hi - lo > 1) {
      const uint32_t mid = (lo + hi) >> 1;
      if (st.g_item0[mid] <= i) lo = mid; else hi = mid;
    }
    const uint32_t g = lo, k = i - st.g_item0[g];
    const uint32_t R = st.gR[g], W = st.gW[g];
    Item it;
    it.group = g;
    if (W <= (uint32_t)kItemCand) {
      const uint32_t rpi = item_rpi(W);
      it.i0 = k * rpi; it.j0 = 0;
      it.nrows = (uint16_t)min(rpi, R - k * rpi); it.nj = (uint16_t)W;
    } else {
      const uint32_t nt2 = (W + kItemCand - 1) / kItemCand;
      it.i0 = k / nt2; it.j0 = (k % nt2) * kItemCand;
      it.nrows = 1; it.nj = (uint16_t)min((uint32_t)kItemCand, W - it.j0);
    }
    st.items[i] = it;
  }
  for (uint32_t u = tid; u < n_units; u += nt) {   // one thread per UNIT: its group
    uint32_t lo = 0, hi = ng;
    while (hi - lo > 1) {
      const uint32_t mid = (lo + hi) >> 1;
      if (st.g_unit0[mid] <= u) lo = mid; else hi = mid;
    }
    st.unit_group[u] = lo;
  }
  // LS: the pre-filter kernel walks rows, not items, so the pass-bit masks are cleared here
  if (stage == S_LS)
    for (size_t w = tid; w < (size_t)n_items * kItemWords; w += nt) st.mask[w] = 0;
}

// ------------------------------------------------------------------ per-item pass counts from the masks
// One warp per item (stages whose decide kernel sets the mask bits with global atomics).
__global__ void __launch_bounds__(256) k_item_counts(SlotDev s, int stage) {
  const StageBuf &st = s.st[stage];
  const uint32_t n = s.hdr->n_items[stage];
  const int lane = threadIdx.x & 31;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
  for (uint32_t it = warp; it < n; it += nwarp) publish_item(st, it, st.mask[(size_t)it * kItemWords + lane]);
}
void launch_item_counts(const Ctx &c, const SlotDev &s, int stage, cudaStream_t st) {
  static const char *const nm[S_NSTAGE] = {"k_item_counts[MD]", "k_item_counts[LS]", "k_item_counts[T3]",
                                           "k_item_counts[T5]", "k_item_counts[pT5]", "k_item_counts[pT3]"};
  k_item_counts<<<c.n_sm * 2, 256, 0, st>>>(s, stage); LST_MARK(c, st, nm[stage]);
}

// ------------------------------------------------------------------ scan item pass counts
// One block.  Exact object count of the level; overflow empties the level (never truncates).
__global__ void k_scan_items(SlotDev s, int stage, int level, uint32_t cap) {
  __shared__ uint32_t sh[33];
  Header *hdr = s.hdr;
  const StageBuf &st = s.st[stage];
  const uint32_t n = hdr->n_items[stage];
  const uint32_t chunk = (n + blockDim.x - 1) / blockDim.x;
  const uint32_t b0 = min(n, threadIdx.x * chunk), b1 = min(n, b0 + chunk);
  uint32_t sum = 0;
  for (uint32_t i = b0; i < b1; ++i) sum += st.item_cnt[i];
  uint32_t carry;
  uint32_t run = block_excl_scan(sum, sh, &carry);
  for (uint32_t i = b0; i < b1; ++i) { st.item_base[i] = run; run += st.item_cnt[i]; }
  if (threadIdx.x == 0) {
    if (carry > cap) {
      atomicOr(&hdr->err, (uint32_t)ERR_CAP_OBJ);
      hdr->n_items[stage] = 0;
      hdr->n_obj[level] = 0;
    } else {
      hdr->n_obj[level] = carry;
    }
  }
}

// ------------------------------------------------------------------ row offsets from sorted row keys
// off[r] = first object whose row key >= r, r in [0, n_rows]; keys ascending.
// KIND 0: MD -> module (n_rows = n_modules); 1: LS -> inner MD; 2: T3 -> first MD; 3: T5 -> first MD
// (n_rows = n_md); 4: pT5 -> seed; 5: pT3 -> seed (n_rows = n_seeds)
template <int KIND>
__global__ void k_row_offsets(GeoDev geo, SlotDev s) {
  const Header *hdr = s.hdr;
  uint32_t n, n_rows;
  uint32_t *off;
  if (KIND == 0) { n = hdr->n_obj[0]; n_rows = geo.n_modules; off = s.md_mod_off; }
  else if (KIND == 1) { n = hdr->n_obj[1]; n_rows = hdr->n_obj[0]; off = s.ls_md_off; }
  else if (KIND == 2) { n = hdr->n_obj[2]; n_rows = hdr->n_obj[0]; off = s.t3_md_off; }
  else if (KIND == 3) { n = hdr->n_obj[3]; n_rows = hdr->n_obj[0]; off = s.t5_md_off; }
  else if (KIND == 4) { n = hdr->n_obj[5]; n_rows = hdr->n_seeds; off = s.pt5_pls_off; }
  else { n = hdr->n_obj[4]; n_rows = hdr->n_seeds; off = s.pt3_pls_off; }
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nt = gridDim.x * blockDim.x;
  // one thread per ROW: lower bound of r in the ascending keys (gaps between keys can be thousands
  // of rows wide, e.g. outer-layer MDs start no T3 / T5)
  for (uint32_t r = tid; r <= n_rows; r += nt) {
    uint32_t lo = 0, hi = n;           // first k in [0, n] with key[k] >= r
    while (lo < hi) {
      const uint32_t mid = (lo + hi) >> 1;
      uint32_t key;
      if (KIND == 0) key = s.md_mod[mid] >> 2;
      else if (KIND == 1) key = s.ls_md[mid].x;
      else if (KIND == 2) key = s.t3_md[mid].x;
      else if (KIND == 3) key = s.t5_md[5 * (size_t)mid];
      else if (KIND == 4) key = s.pt5_po[mid].x;
      else key = s.pt3_po[mid].x;
      if (key < r) lo = mid + 1; else hi = mid;
    }
    off[r] = lo;
  }
}

// ------------------------------------------------------------------ host launchers
static inline int grid_for(uint32_t n, int threads, int max_blocks) {
  long b = ((long)n + threads - 1) / threads;
  if (b < 1) b = 1;
  if (b > max_blocks) b = max_blocks;
  return (int)b;
}

void launch_index(const Ctx &c, const SlotDev &s, cudaStream_t st) {
  cudaMemsetAsync(s.det_cnt, 0, sizeof(uint32_t) * (c.geo.n_det + 1), st);
  k_begin<<<1, 32, 0, st>>>(s); LST_MARK(c, st, "k_begin");
  const int g = grid_for(s.cap_hits, 256, c.n_sm * 8);
  k_hist<<<g, 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_hist");
  k_det_scan<<<1, 1024, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_det_scan");
  k_scatter<<<g, 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_scatter");
  k_rank<<<g, 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_rank");
}

static const char *const kEmitName[S_NSTAGE] = {"k_emit_items[MD]", "k_emit_items[LS]", "k_emit_items[T3]",
                                                  "k_emit_items[T5]", "k_emit_items[pT5]", "k_emit_items[pT3]"};
static const char *const kEmitFillName[S_NSTAGE] = {"k_emit_fill[MD]", "k_emit_fill[LS]", "k_emit_fill[T3]",
                                                      "k_emit_fill[T5]", "k_emit_fill[pT5]", "k_emit_fill[pT3]"};
static const char *const kScanName[S_NSTAGE] = {"k_scan_items[MD]", "k_scan_items[LS]", "k_scan_items[T3]",
                                                  "k_scan_items[T5]", "k_scan_items[pT5]", "k_scan_items[pT3]"};
void launch_emit(const Ctx &c, const SlotDev &s, int stage, int rows_level, cudaStream_t st) {
  k_emit_items<<<1, 1024, 0, st>>>(s, stage, rows_level); LST_MARK(c, st, kEmitName[stage]);
  k_emit_fill<<<c.n_sm, 256, 0, st>>>(s, stage); LST_MARK(c, st, kEmitFillName[stage]);
}
void launch_scan_items(const Ctx &c, const SlotDev &s, int stage, int level, uint32_t cap, cudaStream_t st) {
  k_scan_items<<<1, 1024, 0, st>>>(s, stage, level, cap); LST_MARK(c, st, kScanName[stage]);
}
void launch_row_offsets(const Ctx &c, const SlotDev &s, int kind, cudaStream_t st) {
  const uint32_t rows[6] = {c.geo.n_modules, s.cap_md, s.cap_md, s.cap_md, s.cap_seeds, s.cap_seeds};
  const int g = grid_for(rows[kind] + 1, 256, c.n_sm * 4);
  switch (kind) {
    case 0: k_row_offsets<0><<<g, 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_row_offsets[MD]"); break;
    case 1: k_row_offsets<1><<<g, 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_row_offsets[LS]"); break;
    case 2: k_row_offsets<2><<<g, 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_row_offsets[T3]"); break;
    case 3: k_row_offsets<3><<<g, 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_row_offsets[T5]"); break;
    case 4: k_row_offsets<4><<<g, 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_row_offsets[pT5]"); break;
    default: k_row_offsets<5><<<g, 256, 0, st>>>(c.geo, s); LST_MARK(c, st, "k_row_offsets[pT3]"); break;
  }
}

// ------------------------------------------------------------------ device-wide exclusive scan
// out[0..n) = exclusive prefix of in[0..n), out[n] = total; n = *n_ptr (a Header field).  Two
// launches of kScanBlocks blocks: per-block sums (the last block to finish scans them), then the
// per-block scan with its carry.  in == out is allowed.  part: kScanBlocks + 2 words, last = ticket.
__global__ void __launch_bounds__(kScanThreads) k_scan_sums(const uint32_t *in, const uint32_t *n_ptr, uint32_t *part) {
  __shared__ uint32_t sh[33];
  __shared__ bool last;
  const uint32_t n = *n_ptr;
  const uint32_t chunk = (n + gridDim.x - 1) / gridDim.x;
  const uint32_t b0 = min(n, blockIdx.x * chunk), b1 = min(n, b0 + chunk);
  uint32_t sum = 0;
  for (uint32_t i = b0 + threadIdx.x; i < b1; i += blockDim.x) sum += in[i];
  uint32_t tot;
  block_excl_scan(sum, sh, &tot);
  if (threadIdx.x == 0) {
    part[blockIdx.x] = tot;
    __threadfence();
    last = atomicAdd(&part[kScanBlocks + 1], 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  const uint32_t v = threadIdx.x < gridDim.x ? __ldcg(&part[threadIdx.x]) : 0u;
  const uint32_t e = block_excl_scan(v, sh, &tot);
  if (threadIdx.x < gridDim.x) part[threadIdx.x] = e;
  if (threadIdx.x == 0) { part[kScanBlocks] = tot; part[kScanBlocks + 1] = 0; }
}
__global__ void __launch_bounds__(kScanThreads) k_scan_apply(const uint32_t *in, const uint32_t *n_ptr, const uint32_t *part,
                                                             uint32_t *out) {
  __shared__ uint32_t sh[33];
  const uint32_t n = *n_ptr;
  const uint32_t chunk = (n + gridDim.x - 1) / gridDim.x;
  const uint32_t b0 = min(n, blockIdx.x * chunk), b1 = min(n, b0 + chunk);
  uint32_t carry = part[blockIdx.x];
  for (uint32_t base = b0; base < b1; base += blockDim.x) {
    const uint32_t i = base + threadIdx.x;
    const uint32_t v = i < b1 ? in[i] : 0u;
    uint32_t tot;
    const uint32_t e = block_excl_scan(v, sh, &tot);
    if (i < b1) out[i] = carry + e;
    carry += tot;
    __syncthreads();
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = part[kScanBlocks];
}
void launch_scan(const Ctx &c, const SlotDev &s, const uint32_t *in, uint32_t *out, const uint32_t *n_ptr,
                 cudaStream_t st) {
  k_scan_sums<<<kScanBlocks, kScanThreads, 0, st>>>(in, n_ptr, s.scan_part); LST_MARK(c, st, "k_scan_sums");
  k_scan_apply<<<kScanBlocks, kScanThreads, 0, st>>>(in, n_ptr, s.scan_part, out); LST_MARK(c, st, "k_scan_apply");
}

}  // namespace lst
