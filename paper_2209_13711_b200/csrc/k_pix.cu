// k_pix.cu -- a5 pixel-seeded pT5 / pT3 (Fig. 10-11; reading C6).
//
// The definition is "all (pixel seed, T5 / T3) pairs".  The enumeration is restricted, without
// changing the result, to the objects whose FIRST anchor can pass its two residual cuts: per seed
// the start-layer modules whose lower-sensor box (lst_geometry) overlaps the seed's extrapolation
// window are listed (k_px_modules); the (seed, module) pairs are the rows of the generic join
// (k_t3t5.cu), whose right lists are the T5 / T3 starting in that module.  The window test is
// conservative (interval arithmetic on the box plus margins); tests compare with the oracle's
// brute force.
#include <algorithm>

#include "lst_launch.h"

namespace lst {

constexpr float kPxMarginPhi = 2e-3f;   // rad, added to every azimuthal window
constexpr float kPxMarginLen = 5e-2f;   // cm, added to every z / r window

__device__ __forceinline__ float asin_sat(float v) { return asinf(fminf(1.0f, fmaxf(-1.0f, v))); }

__device__ __forceinline__ float wrap_f(float d) {   // to [-pi, pi]; error ~1e-7 |d|, far below kPxMarginPhi
  return d - 6.2831853071795864769f * rintf(d * 0.15915494309189533577f);
}

// Can a hit inside a ROW of start modules (same box up to phic) pass the first-anchor cuts of seed
// (kp, sinh eta, phi, z0)?  Everything except the module's phic is decided here; for a compatible
// row the azimuthal window |wrap(phic - *centre)| <= *halfw selects its modules.
// r1 = {hphi, rmin, rmax, category}, r2 = {zmin, zmax, sig_t / rmin, -}.
__device__ __forceinline__ bool px_row_window(const Params &g, float4 r1, float4 r2, float kp, float sh, float phi,
                                              float z0, float *centre, float *halfw) {
  const int cat = (int)r1.w;
  const float hphi = r1.x, rlo = r1.y, rhi = r1.z, zlo = r2.x, zhi = r2.y;
  const float akp = fabsf(kp);
  const float sgn = kp < 0.0f ? -1.0f : 1.0f;
  const float ns = g.f_ns;
  if (cat < 2) {
    // barrel: arc length s(r) = asin(|k| r) / |k| is increasing in r
    const float a_lo = asin_sat(akp * rlo), a_hi = asin_sat(akp * rhi);
    const float s_lo = akp * rlo <= 1e-4f ? rlo : a_lo / akp, s_hi = akp * rhi <= 1e-4f ? rhi : a_hi / akp;
    const float sgp = (float)g.seed_sig_phi + (float)g.seed_sig_pt * akp * s_hi + r2.z;
    *centre = phi + sgn * 0.5f * (a_lo + a_hi);
    *halfw = hphi + 0.5f * (a_hi - a_lo) + ns * sgp + kPxMarginPhi;
    const float z1 = z0 + sh * s_lo, z2 = z0 + sh * s_hi;
    const float tol = ns * ((float)g.seed_sig_z + g.f_sig_z[cat]) + kPxMarginLen + 1e-3f * (fabsf(z1) + fabsf(z2));
    return fmaxf(z1, z2) + tol >= zlo && fminf(z1, z2) - tol <= zhi;
  }
  // endcap: the anchor's z is the lower-sensor plane, so the arc length is known
  if (!(fabsf(sh) > 1e-9f)) return false;
  const float al = (zlo - z0) / sh;
  if (!(al > 0.0f)) return false;
  const float sgp = (float)g.seed_sig_phi + (float)g.seed_sig_pt * akp * al + r2.z;
  *centre = phi + kp * al;
  *halfw = hphi + ns * sgp + kPxMarginPhi + 1e-3f * akp * al;
  const float ka = kp * al;
  const float rp = fabsf(ka) <= 1e-4f ? al : sinf(ka) / kp;
  const float tol = ns * ((float)g.seed_sig_z / fabsf(sh) + g.f_sig_r[cat]) + kPxMarginLen + 1e-3f * fabsf(rp);
  return rp + tol >= rlo && rp - tol <= rhi;
}

// ------------------------------------------------------------------ seed lookups of the cleaning (reading C7)
// "Seeds a and b share a pixel hit" is looked up through the pixel-hit ids themselves: every id is
// inserted into a hash set (linear probing; at most half full), and a seed remembers the slots of its
// 4 ids.  Flags per slot (pid_has5 / pid_has3) then answer "does some seed with a surviving pT5 /
// pT3 contain this pixel hit" without any seed-to-seed list.
__device__ __forceinline__ uint32_t pid_hash(uint32_t id) { return (id * 0x9E3779B1u) ^ (id >> 15); }
__device__ __forceinline__ void pid_insert(const SlotDev &s, uint32_t i) {
  const uint32_t id = s.seed_ids[i], mask = s.pid_size - 1;
  const unsigned long long key = (1ull << 32) | id;
  uint32_t h = pid_hash(id) & mask;
  for (;;) {
    const unsigned long long old = atomicCAS(&s.pid_key[h], 0ull, key);
    if (old == 0ull || old == key) break;
    h = (h + 1) & mask;
  }
  s.pls_slot[i] = h;
}

// Last block of the seed-preparation kernel: offsets of the per-seed (seed, module) lists and their
// total (0 + error flag if the rows do not fit), offsets of the eta bins (counted by the seeds' warps).
__device__ void seed_epilogue(const SlotDev &s) {
  __shared__ uint32_t sh[33];
  Header *hdr = s.hdr;
  const uint32_t n = hdr->n_seeds;
  block_scan_array(s.px_cnt, s.px_off, n, sh);
  block_scan_array(s.pls_bin_cnt, s.pls_bin_off, (uint32_t)kEtaBins, sh);
  if (threadIdx.x == 0) {
    uint32_t tot = s.px_off[n];
    if (tot > s.cap_seeds * (uint32_t)kPxCap) { atomicOr(&hdr->err, (uint32_t)ERR_CAP_PIX); tot = 0; }
    hdr->n_obj[kPairLevel] = tot;
  }
}

static inline size_t px_shared_bytes(const Ctx &c) {   // 8 warps x (>= 64 words: the queue of the fill pass)
  return 8 * std::max<size_t>((size_t)(c.geo.n_start + 31) / 32, 64) * sizeof(uint32_t);
}
static inline int px_grid(const Ctx &c, const Batch &b) {
  int g = (int)((b.s[0].cap_seeds + 7) / 8);
  return g > c.n_sm * 8 ? c.n_sm * 8 : (g < 1 ? 1 : g);
}

// One warp per seed.  FILL = false: one bit per (seed, start module): the lanes test the module
// ROWS (32 at a time); for every compatible row the warp walks the row's modules and keeps those
// inside the azimuthal window.  FILL = true: expand the bits into the (seed, module) rows at the
// seed's offset, modules ascending.  (A seed with eta ~ 0 is compatible with every endcap module of
// a side - its extrapolation tolerances diverge - so the lists are sized exactly, not capped per
// seed.)  Dynamic shared memory: 8 warps x nw words of bits.
template <bool FILL>
__global__ void __launch_bounds__(256, FILL ? 6 : 5) k_px_modules(const __grid_constant__ GeoDev geo, const __grid_constant__ Batch B,
                                                     const __grid_constant__ Params g) {
  extern __shared__ uint32_t px_sh[];
  pdl_enter();
  LST_SLOT(B);
  const uint32_t n_seeds = s.hdr->n_seeds;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
  const uint32_t nw = (geo.n_start + 31) / 32;
  const bool have_rows = s.hdr->n_obj[kPairLevel] != 0;      // 0: no compatible module at all, or the rows overflowed
  uint32_t *wbits = px_sh + (size_t)wib * (nw > 64u ? nw : 64u);
  for (uint32_t p = warp; p < n_seeds; p += nwarp) {
    uint32_t *bits = s.px_bits + (size_t)p * nw;
    if (FILL) {
      if (lane == 0) {      // the seed into its eta bin (the order inside a bin is irrelevant)
        const int bin = eta_bin(g, (double)s.seed_eta[p]);
        s.pls_bin_ent[s.pls_bin_off[bin] + atomicAdd(&s.pls_bin_cur[bin], 1u)] = p;
      }
      if (!have_rows) continue;
      const float pt = s.seed_pt[p], phi = s.seed_phi[p], z0 = s.seed_z0[p];
      const float kp = -(float)s.seed_q[p] * (float)g.kB / (2.0f * pt);
      const float sh = sinhf(s.seed_eta[p]);
      // the set bits (ascending module) go through a warp queue so that the windows of 32 (seed,
      // module) rows are computed at a time
      uint32_t pos = s.px_off[p];
      WarpQueue Q;
      Q.init(wbits);                  // 64 words of this warp's shared area (nw >= 64 is not needed: see launch)
      for (uint32_t wb = 0; wb <= nw; wb += 32) {
        // 32 words at a time, only the non-empty ones are expanded (a seed reaches ~6 of 2 588 modules)
        const uint32_t myw = wb + lane < nw ? bits[wb + lane] : 0u;
        uint32_t nz = __ballot_sync(0xffffffffu, myw != 0u);
        const bool last = wb + 32 > nw;
        // expand the next non-empty word until 32 rows are queued (or the seed is finished), then drain
        for (;;) {
          if (!(Q.n >= 32u || (last && nz == 0u && Q.n > 0u))) {
            if (nz == 0u) break;
            const int src = __ffs(nz) - 1;
            nz &= nz - 1;
            const uint32_t b = __shfl_sync(0xffffffffu, myw, src);
            Q.push(((b >> lane) & 1u) != 0u, (wb + src) * 32 + lane);
            continue;
          }
          const uint32_t take = Q.n < 32u ? Q.n : 32u;
          uint32_t k;
          if (Q.pop(&k)) {
            const uint32_t m = geo.start_mods[k], r = geo.prow_of[k];
            // the row's window again, now for the azimuth of a first anchor instead of the module
            // centre: the module's half width drops out
            float centre = 0.0f, halfw = 0.0f;
            const float4 r1 = geo.prow_b1[r];
            px_row_window(g, r1, geo.prow_b2[r], kp, sh, phi, z0, &centre, &halfw);
            s.px_pair[pos + lane] = make_uint2(p, m);
            // MDs ascend in azimuth (relative to the module centre) inside a module: those inside the
            // window are a range, found here once per row by two binary searches
            uint32_t md0 = s.md_mod_off[m], md1 = s.md_mod_off[m + 1];
            const float wc = wrap_f(centre - geo.phic[m]), ww = halfw - r1.x + 1e-4f;
            if (ww < 2.5f) {      // wider windows wrap around: keep the whole module
              const float lo = wc - ww, hi = wc + ww;
              uint32_t a = md0, b = md1;
              while (a < b) { const uint32_t mid = (a + b) >> 1; if (s.md_prel[mid] < lo) a = mid + 1; else b = mid; }
              const uint32_t first = a;
              b = md1;
              while (a < b) { const uint32_t mid = (a + b) >> 1; if (s.md_prel[mid] <= hi) a = mid + 1; else b = mid; }
              md0 = first; md1 = a;
            }
            s.px_rng[pos + lane] = make_uint2(md0, md1);
          }
          pos += take;
        }
      }
      __syncwarp();
    } else {
      const float pt = s.seed_pt[p], phi = s.seed_phi[p], z0 = s.seed_z0[p];
      const float kp = -(float)s.seed_q[p] * (float)g.kB / (2.0f * pt);
      const float sh = sinhf(s.seed_eta[p]);
      if (lane == 0 && !(fabsf(pt) <= 3.0e38f && fabsf(s.seed_eta[p]) <= 3.0e38f && fabsf(phi) <= 3.0e38f && fabsf(z0) <= 3.0e38f))
        atomicOr(&s.hdr->err, (uint32_t)ERR_NONFINITE);
      for (uint32_t w = lane; w < nw; w += 32) wbits[w] = 0;
      __syncwarp();
      for (uint32_t rb = 0; rb < geo.n_prow; rb += 32) {
        const uint32_t r = rb + lane;
        float centre = 0.0f, halfw = 0.0f;
        bool ok = false;
        if (r < geo.n_prow && pt > 0.0f) ok = px_row_window(g, geo.prow_b1[r], geo.prow_b2[r], kp, sh, phi, z0, &centre, &halfw);
        uint32_t live = __ballot_sync(0xffffffffu, ok);
        while (live) {                                   // warp-uniform loop over the compatible rows
          const int src = __ffs(live) - 1;
          live &= live - 1;
          const float c = __shfl_sync(0xffffffffu, centre, src), hw = __shfl_sync(0xffffffffu, halfw, src);
          const uint32_t m0 = geo.prow_off[rb + src], m1 = geo.prow_off[rb + src + 1];
          for (uint32_t m = m0 + lane; m < m1; m += 32) {
            if (!(fabsf(wrap_f(geo.prow_phic[m] - c)) > hw)) {
              const uint32_t k = geo.prow_k[m];
              atomicOr(&wbits[k >> 5], 1u << (k & 31));
            }
          }
        }
      }
      __syncwarp();
      uint32_t cnt = 0;
      for (uint32_t w = lane; w < nw; w += 32) {
        const uint32_t b = wbits[w];
        bits[w] = b;
        cnt += __popc(b);
      }
      cnt = warp_sum(cnt);
      if (lane == 0) s.px_cnt[p] = cnt;
      if (lane < 4) pid_insert(s, 4 * p + lane);
      if (lane == 4) atomicAdd(&s.pls_bin_cnt[eta_bin(g, (double)s.seed_eta[p])], 1u);
      __syncwarp();
    }
  }
  if (!FILL) {
    if (!last_block(&s.hdr->ticket[TK_SEEDS], gridDim.x)) return;
    seed_epilogue(s);
  }
}

void launch_seed_prep(const Ctx &c, const Batch &b, cudaStream_t st, bool first) {
  const size_t shb = px_shared_bytes(c);
  if (shb > 48 * 1024) cudaFuncSetAttribute(k_px_modules<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shb);
  launch_k(c, st, "k_px_modules<false>", k_px_modules<false>, dim3(px_grid(c, b)), 256, shb, first, c.geo, b, c.par);
}
void launch_seed_rows(const Ctx &c, const Batch &b, cudaStream_t st) {
  const size_t shb = px_shared_bytes(c);
  if (shb > 48 * 1024) cudaFuncSetAttribute(k_px_modules<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shb);
  launch_k(c, st, "k_px_modules<true>", k_px_modules<true>, dim3(px_grid(c, b)), 256, shb, false, c.geo, b, c.par);
}

}  // namespace lst
