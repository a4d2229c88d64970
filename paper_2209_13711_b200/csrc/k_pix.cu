// k_pix.cu -- a5 pixel-seeded pT5 / pT3 (Fig. 10-11; reading C6).
#include "lst_launch.h"

namespace lst {
void launch_pixel(const Ctx &c, const SlotDev &s, cudaStream_t st) { (void)c; (void)s; (void)st; }
}  // namespace lst
