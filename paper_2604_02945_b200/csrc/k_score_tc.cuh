// k_score_tc.cuh — tcgen05 / TMA fast path of the score pass (placeholder until the kernel lands: disabled).
#pragma once
#include "../../include/msas.h"
#include "msas_internal.cuh"

namespace msas {
struct TcSchedule { bool enabled = false; };
inline size_t tc_schedule_bytes(const mas_segment*, int32_t) { return 0; }
inline void tc_build_schedule(TcSchedule& t, const mas_segment*, int32_t, const int64_t*, int32_t, int32_t, int, char*, char*) { t.enabled = false; }
inline void tc_set_kernel_attrs() {}
inline int tc_launch_score(const TcSchedule&, const void*, const void*, float*, float*, float*, float*, int64_t, int64_t, int, cudaStream_t) { return -1; }
}  // namespace msas
