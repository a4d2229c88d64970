// k_common.cu -- a0 hit indexing (PAPER.md:125 SoA event data) and the generic
// work-list kernels (per-item pass counts + exact sizes, device-wide scan) used by every stage.
#include "lst_launch.h"

namespace lst {

// ------------------------------------------------------------------ a0.1 histogram of det ids (+ a0.2 in the last block)
// Every hit takes its arrival rank inside its det (the order is made canonical by k_rank) and is
// validated (include/lst.h): finite coordinates; a lower-sensor hit inside its module's box (the
// dead-edge pruning of lst_create and the pixel-seed windows rely on the boxes).
// Last block: det_off = exclusive scan of det_cnt; the MD groups (module m: rows = lower hits,
// width = upper hits), their work items and the MD candidate count.
__global__ void __launch_bounds__(1024) k_hist(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B) {
  __shared__ uint32_t sh[33];
  __shared__ unsigned long long sh_cand;
  pdl_enter();
  LST_SLOT(B);
  Header *hdr = s.hdr;
  const uint32_t n = hdr->n_hits;
  for (uint32_t h = blockIdx.x * blockDim.x + threadIdx.x; h < n; h += gridDim.x * blockDim.x) {
    const uint32_t d = s.raw_det[h];
    if (d >= geo.n_det) { atomicOr(&hdr->err, (uint32_t)ERR_DET); continue; }
    s.tmp_slot[h] = atomicAdd(&s.det_cnt[d], 1u);
    const float x = s.raw_x[h], y = s.raw_y[h], z = s.raw_z[h];
    if (!(fabsf(x) <= 3.0e38f && fabsf(y) <= 3.0e38f && fabsf(z) <= 3.0e38f)) { atomicOr(&hdr->err, (uint32_t)ERR_NONFINITE); continue; }
    if ((d & 1u) == 0u) {
      const uint32_t m = d >> 1;
      const float r = sqrtf(x * x + y * y);
      const float dp = atan2f(y, x) - geo.phic[m];
      const float dphi = fabsf(dp - 6.2831853071795864769f * rintf(dp * 0.15915494309189533577f));
      const bool in = r >= geo.rmin[m] - kBoxTolLen && r <= geo.rmax[m] + kBoxTolLen && z >= geo.zmin[m] - kBoxTolLen &&
                      z <= geo.zmax[m] + kBoxTolLen && dphi <= geo.hphi[m] + kBoxTolPhi + 4e-7f * (fabsf(geo.phic[m]) + 3.2f);
      if (!in) atomicOr(&hdr->err, (uint32_t)ERR_BOX);
    }
  }
  if (!last_block(&hdr->ticket[TK_HIST], gridDim.x)) return;
  block_scan_array(s.det_cnt, s.det_off, geo.n_det, sh);
  const StageBuf &st = s.st[S_MD];
  if (threadIdx.x == 0) sh_cand = 0ull;
  __syncthreads();
  // two modules (four dets: one uint4 of det_cnt) per thread and round; one block scan per round
  const uint32_t ng = geo.n_modules;
  uint32_t carry = 0, rcarry = 0;
  unsigned long long my_cand = 0;
  for (uint32_t base = 0; base < ng; base += 2 * blockDim.x) {
    const uint32_t m = base + 2 * threadIdx.x;
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (m + 1 < ng) v = __ldcg(reinterpret_cast<const uint4 *>(s.det_cnt + 2 * m));
    else if (m < ng) { v.x = __ldcg(&s.det_cnt[2 * m]); v.y = __ldcg(&s.det_cnt[2 * m + 1]); }
    const uint32_t i0 = items_of(v.x, v.y), i1 = items_of(v.z, v.w);
    uint32_t tot;
    const uint32_t e = carry + block_excl_scan(i0 + i1, sh, &tot);
    if (m < ng) { st.gR[m] = v.x; st.gW[m] = v.y; st.g_item0[m] = e; }
    if (m + 1 < ng) { st.gR[m + 1] = v.z; st.gW[m + 1] = v.w; st.g_item0[m + 1] = e + i0; }
    my_cand += (unsigned long long)v.x * v.y + (unsigned long long)v.z * v.w;
    carry += tot;
    __syncthreads();
    uint32_t rtot;                                                     // rows (lower-sensor hits) before the module
    const uint32_t re = rcarry + block_excl_scan(v.x + v.z, sh, &rtot);
    if (m < ng) s.md_row0[m] = re;
    if (m + 1 < ng) s.md_row0[m + 1] = re + v.x;
    rcarry += rtot;
    __syncthreads();
  }
  const uint32_t total = carry;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) my_cand += __shfl_xor_sync(0xffffffffu, my_cand, o);
  if ((threadIdx.x & 31) == 0 && my_cand) atomicAdd(&sh_cand, my_cand);
  __syncthreads();
  if (threadIdx.x == 0) {
    const bool overflow = total > st.cap_items;
    st.g_item0[ng] = total;
    s.md_row0[ng] = rcarry;
    hdr->n_groups[S_MD] = ng;
    hdr->n_items[S_MD] = overflow ? 0u : total;
    hdr->cand[S_MD] = sh_cand;
    hdr->n_inc = 3u * n;
    if (overflow) atomicOr(&hdr->err, (uint32_t)ERR_CAP_ITEMS);
  }
}

// ------------------------------------------------------------------ a0.3 scatter (unordered within a det)
__global__ void __launch_bounds__(256) k_scatter(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B) {
  pdl_enter();
  LST_SLOT(B);
  const uint32_t n = s.hdr->n_hits;
  for (uint32_t h = blockIdx.x * blockDim.x + threadIdx.x; h < n; h += gridDim.x * blockDim.x) {
    const uint32_t d = s.raw_det[h];
    if (d >= geo.n_det) continue;
    const uint32_t p = s.det_off[d] + s.tmp_slot[h];
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
__global__ void __launch_bounds__(256) k_rank(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B) {
  pdl_enter();
  LST_SLOT(B);
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
    if ((d & 1u) == 0u) s.row_mod[s.md_row0[d >> 1] + r] = d >> 1;   // MD row -> module (k_md_eval: one thread per row)
  }
}

void launch_index(const Ctx &c, const Batch &b, cudaStream_t st) {
  const uint32_t nh = b.s[0].cap_hits;
  launch_k(c, st, "k_hist", k_hist, dim3(grid_for(nh, 1024, c.n_sm * 2)), 1024, 0, true, c.geo, b);
  const int g = grid_for(nh, 256, c.n_sm * 8);
  launch_k(c, st, "k_scatter", k_scatter, dim3(g), 256, 0, false, c.geo, b);
  launch_k(c, st, "k_rank", k_rank, dim3(g), 256, 0, false, c.geo, b);
}

// ------------------------------------------------------------------ per-item pass counts + exact sizes
// Block b owns the items [b C, (b + 1) C): a warp per item turns the item's mask words into running
// counts (wpre) and its pass count; the block scans its items' counts; the last block to finish scans
// the per-block sums, completes item_base and publishes the level's exact size (an overflow empties
// the level, it never truncates).  blockIdx.y selects the stage when two stages share the launch
// (pT5 / pT3: stage0 + y, level0 - y, caps cap0 / cap1).
__global__ void __launch_bounds__(kCountThreads) k_counts(const __grid_constant__ Batch B, int stage0, int level0, uint32_t cap0,
                                                           uint32_t cap1) {
  __shared__ uint32_t sh[33];
  pdl_enter();
  LST_SLOT(B);
  const int stage = stage0 + (int)blockIdx.y, level = level0 - (int)blockIdx.y;
  const uint32_t cap = blockIdx.y ? cap1 : cap0;
  Header *hdr = s.hdr;
  const StageBuf &st = s.st[stage];
  const uint32_t n = hdr->n_items[stage];
  const uint32_t C = (n + gridDim.x - 1) / gridDim.x;
  const uint32_t i0 = min(n, blockIdx.x * C), i1 = min(n, i0 + C);
  const int lane = threadIdx.x & 31;
  for (uint32_t it = i0 + (threadIdx.x >> 5); it < i1; it += kCountThreads / 32) publish_item(st, it, st.mask[(size_t)it * kItemWords + lane]);
  __syncthreads();
  uint32_t carry = 0;
  for (uint32_t base = i0; base < i1; base += blockDim.x) {
    const uint32_t i = base + threadIdx.x;
    const uint32_t v = i < i1 ? st.item_cnt[i] : 0u;
    uint32_t tot;
    const uint32_t e = block_excl_scan(v, sh, &tot);
    if (i < i1) st.item_base[i] = carry + e;
    carry += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) st.cblk[blockIdx.x] = carry;
  if (!last_block(&hdr->ticket[TK_COUNTS + stage], gridDim.x)) return;
  const uint32_t total = lb_scan_parts(st.cblk, gridDim.x, sh);
  lb_add_block_prefix(st.item_base, n, st.cblk, C);
  if (threadIdx.x == 0) {
    if (total > cap) {
      atomicOr(&hdr->err, (uint32_t)ERR_CAP_OBJ);
      hdr->n_items[stage] = 0;
      hdr->n_obj[level] = 0;
    } else {
      hdr->n_obj[level] = total;
    }
  }
}
// ------------------------------------------------------------------ occupancy truncation
// Optional memory mode: a bucket (MD, LS, T3, T5: the module of the object's first MD; pT3 / pT5: the
// pixel seed) keeps at most K accepted candidates, the K FIRST in canonical order ("the K smallest
// keys": a candidate's key is its position in the enumeration of the method's definition).  A bucket's
// candidates are one contiguous range of pass bits, so the rule is: clear every set bit after the
// K-th one of the range.  One warp per bucket, between the decide kernel and k_counts; sizes stay
// exact (of the truncated set).  K = Params::trunc[level][logical layer of the module] ([level][0]
// for the per-seed caps), 0 = no cap.
__device__ __forceinline__ uint32_t row_key(const StageBuf &st, uint32_t a, uint32_t n_rows, uint32_t n_items) {
  return a < n_rows ? st.g_item0[a / kRowChunk] * (uint32_t)kItemCand + st.row_cum[a] : n_items * (uint32_t)kItemCand;
}
__global__ void __launch_bounds__(256) k_truncate(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B,
                                                   const __grid_constant__ Params g, int stage0) {
  pdl_enter();
  LST_SLOT(B);
  const int stage = stage0 + (int)blockIdx.y;
  const Header *hdr = s.hdr;
  const StageBuf &st = s.st[stage];
  const uint32_t n_items = hdr->n_items[stage];
  if (n_items == 0) return;
  const int level = stage == S_PT5 ? 5 : (stage == S_PT3 ? 4 : stage);
  const bool by_seed = stage >= S_PT5;
  const uint32_t n_buckets = by_seed ? hdr->n_seeds : geo.n_modules;
  const uint32_t n_rows = stage == S_T3 ? hdr->n_obj[1] : (stage == S_T5 ? hdr->n_obj[2] : hdr->n_obj[kPairLevel]);
  const int lane = threadIdx.x & 31;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
  for (uint32_t b = warp; b < n_buckets; b += nwarp) {
    const uint32_t K = by_seed ? g.trunc[level][0] : g.trunc[level][geo.layer[b] & 15];
    if (K == 0) continue;
    uint32_t key_lo, key_hi;
    if (stage <= S_LS) { key_lo = st.g_item0[b] * (uint32_t)kItemCand; key_hi = st.g_item0[b + 1] * (uint32_t)kItemCand; }
    else {
      uint32_t a0, a1;
      if (by_seed) { a0 = s.px_off[b]; a1 = s.px_off[b + 1]; }
      else {
        const uint32_t *off = stage == S_T3 ? s.ls_md_off : s.t3_md_off;
        a0 = off[s.md_mod_off[b]]; a1 = off[s.md_mod_off[b + 1]];
      }
      key_lo = row_key(st, a0, n_rows, n_items); key_hi = row_key(st, a1, n_rows, n_items);
    }
    if (key_lo >= key_hi) continue;
    const uint32_t w_lo = key_lo >> 5, w_hi = (key_hi + 31u) >> 5;     // mask word of a key = key / 32 (kItemCand = 32 words)
    uint32_t running = 0;
    for (uint32_t wb = w_lo; wb < w_hi; wb += 32) {
      const uint32_t w = wb + lane;
      uint32_t mk = w < w_hi ? st.mask[w] : 0u;
      if (w == w_lo) mk &= ~((1u << (key_lo & 31u)) - 1u);
      if (w == (key_hi >> 5) && (key_hi & 31u)) mk &= (1u << (key_hi & 31u)) - 1u;
      const uint32_t c = (uint32_t)__popc(mk);
      uint32_t tot;
      const uint32_t before = running + warp_excl_scan(c, &tot);
      if (c && before + c > K) {
        const uint32_t keepn = K > before ? K - before : 0u;             // the lowest keepn set bits of mk stay
        uint32_t t = mk;
        for (uint32_t k = 0; k < keepn; ++k) t &= t - 1u;
        atomicAnd(&st.mask[w], ~t);                                        // edge words are shared with the neighbouring buckets
      }
      running += tot;
    }
  }
}

void launch_counts(const Ctx &c, const Batch &b, int stage, int level, uint32_t cap, bool pair, cudaStream_t st) {
  if (c.trunc_stages & ((1u << stage) | (pair ? 1u << (stage + 1) : 0u))) {
    const uint32_t nb = stage >= S_PT5 ? b.s[0].cap_seeds : c.geo.n_modules;
    launch_k(c, st, "k_truncate", k_truncate, dim3(grid_for(nb, 8, c.n_sm * 4), pair ? 2 : 1), 256, 0, false, c.geo, b, c.par, stage);
  }
  static const char *const nm[S_NSTAGE] = {"k_counts[MD]", "k_counts[LS]", "k_counts[T3]", "k_counts[T5]", "k_counts[pT5+pT3]", "k_counts[pT3]"};
  const uint32_t cap1 = pair ? b.s[0].cap_pt3 : 0u;
  launch_k(c, st, nm[stage], k_counts, dim3(kCountBlocks, pair ? 2 : 1), kCountThreads, 0, false, b, stage, level, cap, cap1);
}

// ------------------------------------------------------------------ device-wide exclusive scan (incidence rows)
// inc_off[0..n) = exclusive prefix of inc_cnt[0..n), inc_off[n] = total, n = Header::n_inc.  Two
// launches of kScanBlocks blocks: per-block sums (the last block to finish scans them), then the
// per-block scan with its carry.  scan_part: kScanBlocks + 2 words, last = ticket (zeroed per run).
__global__ void __launch_bounds__(kScanThreads) k_scan_sums(const __grid_constant__ Batch B) {
  __shared__ uint32_t sh[33];
  pdl_enter();
  LST_SLOT(B);
  const uint32_t *in = s.inc_cnt;
  uint32_t *part = s.scan_part;
  const uint32_t n = s.hdr->n_inc;
  const uint32_t chunk = (n + gridDim.x - 1) / gridDim.x;
  const uint32_t b0 = min(n, blockIdx.x * chunk), b1 = min(n, b0 + chunk);
  uint32_t sum = 0;
  for (uint32_t i = b0 + threadIdx.x; i < b1; i += blockDim.x) sum += in[i];
  uint32_t tot;
  block_excl_scan(sum, sh, &tot);
  if (threadIdx.x == 0) part[blockIdx.x] = tot;
  if (!last_block(&part[kScanBlocks + 1], gridDim.x)) return;
  const uint32_t v = threadIdx.x < gridDim.x ? __ldcg(&part[threadIdx.x]) : 0u;
  const uint32_t e = block_excl_scan(v, sh, &tot);
  if (threadIdx.x < gridDim.x) part[threadIdx.x] = e;
  if (threadIdx.x == 0) part[kScanBlocks] = tot;
}
__global__ void __launch_bounds__(kScanThreads) k_scan_apply(const __grid_constant__ Batch B) {
  __shared__ uint32_t sh[33];
  pdl_enter();
  LST_SLOT(B);
  const uint32_t *in = s.inc_cnt;
  const uint32_t *part = s.scan_part;
  uint32_t *out = s.inc_off;
  const uint32_t n = s.hdr->n_inc;
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
void launch_scan(const Ctx &c, const Batch &b, int which, cudaStream_t st) {
  (void)which;
  launch_k(c, st, "k_scan_sums", k_scan_sums, dim3(kScanBlocks), kScanThreads, 0, false, b);
  launch_k(c, st, "k_scan_apply", k_scan_apply, dim3(kScanBlocks), kScanThreads, 0, false, b);
}

}  // namespace lst
