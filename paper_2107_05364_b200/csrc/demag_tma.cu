// demag_tma.cu — A4/A7, TMA bulk-tensor pipeline variant (placeholder until the pipeline lands:
// reports MT_ERR_UNIMPLEMENTED so that the dispatcher falls back to the register-streaming kernel).
#include "mt_internal.cuh"

int mt_launch_demag_tma(mt_ctx*, const void*, int, int64_t, int64_t, int64_t, const void*, int64_t,
                        const EpiArgs&) {
  return MT_ERR_UNIMPLEMENTED;
}
