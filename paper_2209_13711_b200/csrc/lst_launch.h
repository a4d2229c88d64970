// lst_launch.h -- host-side view of a context and the per-stage launch functions (one per .cu file).
#pragma once
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
#define LST_MARK(ctx, stream, kname)                                                   \
  do {                                                                                 \
    Recorder *r_ = (ctx).rec;                                                          \
    if (r_ && r_->n < Recorder::kMax) {                                                \
      r_->name[r_->n] = (kname);                                                       \
      ++r_->n;                                                                         \
      if (r_->timed) cudaEventRecord(r_->ev[r_->n], (stream));                         \
    }                                                                                  \
  } while (0)

struct Ctx {             // what the launchers need from a context
  Recorder *rec = nullptr;         // set per call (enqueue_chain works on a copy of the context's Ctx)
  GeoDev geo;
  Params par;
  int n_sm;
  int ls_windows = 1;    // lst_config.enum_pruning bit 1: per-row windows of the LS enumeration
};

// k_common.cu
void launch_index(const Ctx &c, const SlotDev &s, cudaStream_t st);                       // 1 memset + 5 kernels
void launch_emit(const Ctx &c, const SlotDev &s, int stage, int rows_level, cudaStream_t st);
void launch_item_counts(const Ctx &c, const SlotDev &s, int stage, cudaStream_t st);
void launch_scan_items(const Ctx &c, const SlotDev &s, int stage, int level, uint32_t cap, cudaStream_t st);
void launch_row_offsets(const Ctx &c, const SlotDev &s, int kind, cudaStream_t st);
void launch_scan(const Ctx &c, const SlotDev &s, const uint32_t *in, uint32_t *out, const uint32_t *n_ptr,
                 cudaStream_t st);                                                        // 2 kernels
// k_mdls.cu
void launch_md(const Ctx &c, const SlotDev &s, cudaStream_t st);
void launch_ls(const Ctx &c, const SlotDev &s, cudaStream_t st);
// k_t3t5.cu
void launch_t3(const Ctx &c, const SlotDev &s, cudaStream_t st);
void launch_t5(const Ctx &c, const SlotDev &s, cudaStream_t st);
void launch_join(const Ctx &c, const SlotDev &s, int kind, cudaStream_t st);   // 0 T3, 1 T5, 2 pT5, 3 pT3
// k_pix.cu
void launch_pixel(const Ctx &c, const SlotDev &s, cudaStream_t st);
// k_dedup.cu
void launch_dedup(const Ctx &c, const SlotDev &s, cudaStream_t st);
// k_export.cu: gather one level into the export scratch (hit_idx, parents, f)
void launch_export(const Ctx &c, const SlotDev &s, int level, cudaStream_t st);

// number of kernel launches (memsets not counted) each launcher enqueues
constexpr int kLaunchesIndex = 5;

}  // namespace lst
