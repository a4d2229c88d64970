// k_export.cu -- lst_get_objects: gather one level into the caller-facing layout of include/lst.h
// (original hit indices in layer order, parents, four derived floats).  Not on the timed path.
#include "lst_launch.h"

namespace lst {

__device__ __forceinline__ void md_orig_hits(const SlotDev &s, uint32_t md, uint32_t *out) {
  const uint2 h = s.md_hit[md];
  out[0] = s.hit_orig[h.x];
  out[1] = s.hit_orig[h.y];
}

__global__ void k_export(SlotDev s, int level) {
  const uint32_t n = s.hdr->n_obj[level];
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    uint32_t par0 = 0, par1 = 0;
    float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
    switch (level) {
      case 0: {
        md_orig_hits(s, i, s.exp_hits + 2 * (size_t)i);
        par0 = s.md_mod[i] >> 2;
        const double2 k = s.md_kd[i];
        f = make_float4(ld_f(s, s.md_dphi, i), (float)k.x, (float)k.y, 0.f);
        break;
      }
      case 1: {
        const uint2 m = s.ls_md[i];
        md_orig_hits(s, m.x, s.exp_hits + 4 * (size_t)i);
        md_orig_hits(s, m.y, s.exp_hits + 4 * (size_t)i + 2);
        par0 = m.x; par1 = m.y;
        f = ld_f4(s, s.ls_f, i);
        break;
      }
      case 2: {
        const uint4 m = s.t3_md[i];
        md_orig_hits(s, m.x, s.exp_hits + 6 * (size_t)i);
        md_orig_hits(s, m.y, s.exp_hits + 6 * (size_t)i + 2);
        md_orig_hits(s, m.z, s.exp_hits + 6 * (size_t)i + 4);
        const uint2 l = s.t3_ls[i];
        par0 = l.x; par1 = l.y;
        const double2 k = s.t3_kd[i];
        f = make_float4(ld_f(s, s.t3_beta, i), (float)k.x, (float)k.y, 0.f);
        break;
      }
      case 3: {
        for (int q = 0; q < 5; ++q) md_orig_hits(s, s.t5_md[5 * (size_t)i + q], s.exp_hits + 10 * (size_t)i + 2 * q);
        const uint2 t = s.t5_t3[i];
        par0 = t.x; par1 = t.y;
        f = ld_f4(s, s.t5_f, i);
        break;
      }
      case 4: {
        const uint2 po = s.pt3_po[i];
        const uint4 m = s.t3_md[po.y];
        md_orig_hits(s, m.x, s.exp_hits + 6 * (size_t)i);
        md_orig_hits(s, m.y, s.exp_hits + 6 * (size_t)i + 2);
        md_orig_hits(s, m.z, s.exp_hits + 6 * (size_t)i + 4);
        par0 = po.x; par1 = po.y;
        f.x = (float)s.pt3_chi2[i];
        break;
      }
      case 5: {
        const uint2 po = s.pt5_po[i];
        for (int q = 0; q < 5; ++q) md_orig_hits(s, s.t5_md[5 * (size_t)po.y + q], s.exp_hits + 10 * (size_t)i + 2 * q);
        par0 = po.x; par1 = po.y;
        f.x = (float)s.pt5_chi2[i];
        break;
      }
      default: {   // TC: 10 OT hits (padded) + 4 pixel-hit ids
        const uint2 to = s.tc_to[i];
        uint32_t *h = s.exp_hits + 14 * (size_t)i;
        for (int q = 0; q < 14; ++q) h[q] = 0xFFFFFFFFu;
        uint32_t pls = 0xFFFFFFFFu;
        if (to.x == 3) {
          for (int q = 0; q < 5; ++q) md_orig_hits(s, s.t5_md[5 * (size_t)to.y + q], h + 2 * q);
        } else if (to.x == 5) {
          const uint2 po = s.pt5_po[to.y];
          pls = po.x;
          for (int q = 0; q < 5; ++q) md_orig_hits(s, s.t5_md[5 * (size_t)po.y + q], h + 2 * q);
        } else if (to.x == 4) {
          const uint2 po = s.pt3_po[to.y];
          pls = po.x;
          const uint4 m = s.t3_md[po.y];
          md_orig_hits(s, m.x, h); md_orig_hits(s, m.y, h + 2); md_orig_hits(s, m.z, h + 4);
        } else {
          pls = to.y;
        }
        if (pls != 0xFFFFFFFFu) for (int q = 0; q < 4; ++q) h[10 + q] = s.seed_ids[4 * (size_t)pls + q];
        par0 = to.x; par1 = to.y;
        f = s.tc_f[i];
        break;
      }
    }
    s.exp_par[2 * (size_t)i] = par0;
    s.exp_par[2 * (size_t)i + 1] = par1;
    reinterpret_cast<float4 *>(s.exp_f)[i] = f;
  }
}

void launch_export(const Ctx &c, const SlotDev &s, int level, cudaStream_t st) {
  k_export<<<c.n_sm * 4, 256, 0, st>>>(s, level);
}

}  // namespace lst
