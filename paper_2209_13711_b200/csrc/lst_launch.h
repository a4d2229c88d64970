// lst_launch.h -- host-side view of a context and the per-stage launch functions (one per .cu file).
#pragma once
#include <utility>

#include "lst_dev.cuh"

namespace lst {

// Launch recorder: counts the kernels a chain enqueues and, when `timed`, drops a CUDA event after
// each one so that lst_run_timed can report per-kernel durations (bench.py, profiles/).
struct Recorder {
  static constexpr int kMax = 96;
  bool timed = false;
  int n = 0;
  const char *name[kMax];
  cudaEvent_t ev[kMax + 1];   // ev[0] = before the first kernel; created by the owner when timed
};

struct Ctx {             // what the launchers need from a context
  Recorder *rec = nullptr;         // set per call (enqueue_chain works on a copy of the context's Ctx)
  GeoDev geo;
  Params par;
  int n_sm;
  int ls_windows = 1;    // lst_config.enum_pruning bit 1: per-row windows of the LS enumeration
  int pdl = 0;           // launch with programmatic stream serialisation (lst_config.use_pdl)
  int nb = 1;            // slots (events) in the batch: gridDim.z of every launch
  int fix_passes = 0;    // lst_config.s0_fixpoint_passes: extra S0 passes over the T5 collection
  unsigned trunc_stages = 0;   // bit k: stage k has an occupancy cap (k_truncate runs before its k_counts)
};

// One launch of the chain: gridDim.z = events of the batch; with c.pdl the kernel may become resident
// while its predecessor drains (every kernel starts with pdl_enter()).  `first`: the launch follows a
// memset, not a kernel, and is serialised the ordinary way.
template <class... KArgs, class... Args>
inline void launch_k(const Ctx &c, cudaStream_t st, const char *name, void (*kern)(KArgs...), dim3 grid, unsigned block,
                     size_t smem, bool first, Args &&...args) {
  cudaLaunchConfig_t cfg = {};
  grid.z = (unsigned)c.nb;
  cfg.gridDim = grid;
  cfg.blockDim = dim3(block, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  const bool pdl = c.pdl && !first;
  cfg.attrs = pdl ? at : nullptr;
  cfg.numAttrs = pdl ? 1u : 0u;
  cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
  Recorder *r = c.rec;
  if (r && r->n < Recorder::kMax) {
    r->name[r->n] = name;
    ++r->n;
    if (r->timed) cudaEventRecord(r->ev[r->n], st);
  }
}

static inline int grid_for(uint32_t n, int threads, int max_blocks) {
  long b = ((long)n + threads - 1) / threads;
  if (b < 1) b = 1;
  if (b > max_blocks) b = max_blocks;
  return (int)b;
}

// k_common.cu
void launch_index(const Ctx &c, const Batch &b, cudaStream_t st);        // k_hist (+ det scan, MD groups), k_scatter, k_rank
void launch_counts(const Ctx &c, const Batch &b, int stage, int level, uint32_t cap, bool pair, cudaStream_t st);
void launch_scan(const Ctx &c, const Batch &b, int which, cudaStream_t st);   // 0: incidence rows (2 kernels)
// k_mdls.cu
void launch_md(const Ctx &c, const Batch &b, cudaStream_t st);
void launch_ls(const Ctx &c, const Batch &b, cudaStream_t st);
// k_t3t5.cu
void launch_t3(const Ctx &c, const Batch &b, cudaStream_t st);
void launch_t5(const Ctx &c, const Batch &b, cudaStream_t st);
void launch_pixel_joins(const Ctx &c, const Batch &b, cudaStream_t st);  // pT5 and pT3 in the same launches (blockIdx.y)
// k_pix.cu
void launch_seed_prep(const Ctx &c, const Batch &b, cudaStream_t st, bool first);   // needs the seeds only
void launch_seed_rows(const Ctx &c, const Batch &b, cudaStream_t st);    // needs the MDs
// k_dedup.cu
void launch_dedup(const Ctx &c, const Batch &b, cudaStream_t st);
// k_export.cu: gather one level into the export scratch (hit_idx, parents, f)
void launch_export(const Ctx &c, const SlotDev &s, int level, cudaStream_t st);

}  // namespace lst
