// stream.cu -- placeholder until the streaming path lands (next commit).
#include "dedisp_internal.h"
void dedisp_stream_free(dedisp_plan_s*) {}
extern "C" int dedisp_stream_begin(dedisp_plan_t, long long) { return DEDISP_EINVAL; }
extern "C" int dedisp_stream_push(dedisp_plan_t, const int8_t*, long long, float*, long long, long long*) { return DEDISP_EINVAL; }
extern "C" int dedisp_stream_sync(dedisp_plan_t) { return DEDISP_EINVAL; }
extern "C" int dedisp_stream_end(dedisp_plan_t) { return DEDISP_EINVAL; }
