/* im_probe.h - measurement probe, not part of the hot path: what the memory system of the device delivers for accesses at
 * DATA-DEPENDENT addresses, the access pattern that bounds the tick simulation ("what bounds
 * k_sim").  `bench.py` calls it once per run and reports the tick simulation against these ceilings next to the
 * streaming (copy) peak of MEASURED_PEAKS.json.  Lives in its own library (libimprobe.so) so that the boundary of the
 * method (inframind.h) holds nothing but the method.
 */
#ifndef IM_PROBE_H
#define IM_PROBE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* access shapes; every thread touches its own pseudo-random 32-byte sector */
#define IM_PROBE_READ16 0       /* 16-byte load */
#define IM_PROBE_WRITE16 1      /* 16-byte store: half a sector, the memory system fills the rest from DRAM */
#define IM_PROBE_WRITE32 2      /* 32-byte store (one 256-bit instruction): a full sector */
#define IM_PROBE_RMW4 3         /* 4-byte load, then a 4-byte store to the same word */
#define IM_PROBE_SHAPES 4

/* Time `ops_per_thread` rounds of four independent accesses per thread over `n_threads` threads (64 per CTA) on
 * `stream` (a cudaStream_t, may be null) and return the rate in units of 1e9 accesses per second in *gops.
 *   dev_buf, bytes : DEVICE scratch buffer the probe may overwrite (caller-owned); bytes >= 2 * window_bytes
 *   window_bytes   : a warp stays inside one window (a multiple of 32; the tick simulation's warps stay inside their
 *                    32-env block of about 1 MB); windows are picked pseudo-randomly and change every 8 rounds
 * One untimed pass precedes the timed one.  Returns 0, or -1 on a bad argument, -2 on a CUDA error. */
int im_probe_random_access(void *dev_buf, size_t bytes, size_t window_bytes, int shape, uint32_t n_threads, uint32_t ops_per_thread,
                           void *stream, double *gops);

#ifdef __cplusplus
}
#endif
#endif
