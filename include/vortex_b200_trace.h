/*
 * vortex_b200_trace.h -- phase tracing of the libvortex_b200 kernels.  A measurement aid, not part
 * of the paper's method and not part of the hot-path ABI of vortex_b200.h.
 */
#ifndef VORTEX_B200_TRACE_H_
#define VORTEX_B200_TRACE_H_

#include "vortex_b200.h"

/* `kernels` with ONE kind set: that kind's CTA c writes row c.  With several kinds set (a whole step on one time line) the
 * score kernel's rows start at 0, the selection kernels' at 1024, the decode kernels' at 4096. */
#ifdef __cplusplus
extern "C" {
#endif

/* Only a library built with -DVX_TRACE
 * (`python -m paper_2606_06453_b200.build --trace` -> libvortex_b200_trace.so) records anything; the
 * product library returns VX_ERR_UNSUPPORTED.  `buffer` is a DEVICE pointer to max_ctas * 16 int64, owned
 * by the caller and zeroed by it; from the next launch on, every CTA (linear block index < max_ctas) of the
 * kernels named in `kernels` stores %globaltimer nanoseconds at its phase boundaries into its 16 slots
 * (slot 15: SM id; slot meanings: paper_2606_06453_b200/trace.py).  buffer == NULL detaches.  Attach one kind
 * at a time: the kinds share the slot numbering. */
enum { VX_TRACE_SCORE = 1, VX_TRACE_TOPK = 2, VX_TRACE_DECODE = 4 };
vx_status vx_trace_attach(vx_ctx *ctx, void *buffer, int32_t max_ctas, int32_t kernels);

#ifdef __cplusplus
}
#endif
#endif /* VORTEX_B200_TRACE_H_ */
