/* lst_static.h -- the one entry point of liblst_b200.so that never allocates.
 *
 * Who this is for.  The regular API (include/lst.h) allocates in three places: lst_create
 * (cudaMalloc of the detector tables), lst_bind_workspace (graph instantiation) and the first
 * lst_get_objects(copy_to_host = 1) of a slot (cudaMallocHost of the staging buffers).  Some hosts
 * of this library must not do that, for instance
 *   - an online event filter that reserved the whole GPU for its own pool at job start: the driver
 *     heap has nothing left, so a cudaMalloc from a plug-in fails, and even a successful one
 *     synchronises the whole device and stalls the filter's other streams in the middle of a run;
 *   - a module loaded into somebody else's process that is only handed device pointers and has no
 *     right (or no allocator handle) to obtain memory of its own.
 * Such a caller can still run step a0 of the chain -- grouping an event's hits by sensor, the index
 * every later stage reads (SoA event data) -- through
 * lst_index_hits_static below.  The working memory the step needs beyond its inputs and outputs
 * (per-sensor counters, per-hit arrival ranks, the unordered copy and its azimuth keys) lives in a
 * fixed array inside the library image instead of a caller workspace.
 *
 * The price.
 *   - Size limit: an event may hold at most LST_STATIC_MAX_HITS hits on at most LST_STATIC_MAX_DETS
 *     sensors.  Larger sizes are refused with LST_EINVAL and a message; nothing is launched.
 *   - The array (about 3.3 MB) is part of the loaded library: every GPU whose context loads
 *     liblst_b200.so carries it until the process exits, whether or not this call is ever used.
 *   - There is ONE array per GPU, shared by every call and every host thread.  Two calls whose kernels
 *     can overlap on the same GPU (different streams without an ordering event between them, or two
 *     threads) race on it and both results are garbage.  Issue the calls on one stream, or order
 *     them with events.  The array keeps what the previous call left in it; the call itself clears
 *     the part that has to start from zero (the counters), asynchronously on `cuda_stream`.
 *   - First call on a GPU: the call looks up the device address of the array for the GPU that is
 *     current (once per GPU, remembered afterwards).  That look-up may make the CUDA runtime load
 *     the library's device code, so make the first call on each GPU during start-up, with that GPU
 *     current, and before any stream capture is begun.  Later calls only enqueue work.
 *
 * The call uses no cudaMalloc, cudaFree, cudaMallocHost, nor any library routine that allocates, and
 * never synchronises: it enqueues two cudaMemsetAsync (the counters, the n_rejected word) and three kernels.
 */
#ifndef LST_STATIC_H
#define LST_STATIC_H
#include <stddef.h>
#include <stdint.h>

#include "lst.h"

#ifdef __cplusplus
extern "C" {
#endif

#define LST_STATIC_MAX_HITS 262144u /* hits per event the fixed array can index (2^18)           */
#define LST_STATIC_MAX_DETS 65536u  /* sensors (2 per module) the fixed array can count (2^16)   */

/* a0 without a workspace: group the hits of one event by sensor id, in the canonical order of the
 * regular path (inside a sensor the hits ascend in azimuth relative to the module centre,
 * phi(hit) - phic[det / 2] wrapped to (-pi, pi], evaluated in fp32; equal keys by ascending caller
 * index).  All array arguments are DEVICE pointers owned by the caller; inputs are only read.
 *
 *   x, y, z, det  : n_hits each (fp32 cm / uint32 det = 2 * module + sensor); may be NULL if n_hits = 0
 *   phic          : n_dets / 2 module-centre azimuths (lst_geometry.phic, copied to the device by
 *                   the caller); n_dets must be even
 *   det_off  (out): n_dets + 1 words; hits of sensor d occupy [det_off[d], det_off[d + 1]) of the two
 *                   arrays below; det_off[n_dets] = number of hits that were indexed
 *   hit_orig (out): n_hits words: caller index of the hit at each sorted position
 *   hit_xyzr (out): 4 * n_hits floats, 16-byte aligned: x, y, z, sqrt(x^2 + y^2) of the hit at each
 *                   sorted position
 *   n_rejected (out): one word: hits whose det >= n_dets; they are left out of the index (entries
 *                   past det_off[n_dets] of hit_orig / hit_xyzr are not written).  Unlike lst_run this
 *                   call does not check coordinates against the module boxes; a NaN coordinate sorts
 *                   as key 0.
 *   cuda_stream   : a cudaStream_t passed as void*; everything is enqueued there, nothing waits.
 *   errbuf        : HOST buffer of errbuf_len bytes that receives a message when the return value is
 *                   not LST_OK (may be NULL; lst_strerror does not know about this call).
 *
 * Returns LST_OK; LST_EINVAL for a null pointer, odd n_dets, misaligned hit_xyzr, or n_hits /
 * n_dets above the two limits (nothing was enqueued, the outputs are untouched); LST_ECUDA if the
 * address look-up, the memset or a launch failed (the outputs are then undefined). */
int lst_index_hits_static(const float *x, const float *y, const float *z, const uint32_t *det, uint32_t n_hits,
                          const float *phic, uint32_t n_dets, uint32_t *det_off, uint32_t *hit_orig, float *hit_xyzr,
                          uint32_t *n_rejected, void *cuda_stream, char *errbuf, size_t errbuf_len);

#ifdef __cplusplus
}
#endif
#endif
