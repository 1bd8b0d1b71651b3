// Chunked-prefill selection (a7, a7').  Placeholder until the tcgen05 kernel lands: reports unsupported.
#include "sparda_internal.cuh"

int sparda_launch_prefill_select(sparda_ctx*, const void*, const void*, int, int, int, int, int, int32_t*, cudaStream_t) {
    return SPARDA_EUNSUPPORTED;
}
int sparda_launch_prefill_baseline(sparda_ctx*, const void*, const void*, int, int, int, int, int, int32_t*, cudaStream_t) {
    return SPARDA_EUNSUPPORTED;
}
