// k_dedup.cu -- a6 duplicate removal and track candidates (reading C7).
#include "lst_launch.h"

namespace lst {
void launch_dedup(const Ctx &c, const SlotDev &s, cudaStream_t st) { (void)c; (void)s; (void)st; }
}  // namespace lst
