// pipeline.cu -- A6: batched multi-event path (streams + CUDA graphs).  Placeholder until the tiled
// kernels land: the entry points exist and report HOUGH_ERR_UNSUPPORTED.
#include "common.cuh"

struct hough_pipeline { int unused; };

extern "C" int hough_pipeline_create(const hough_binning*, const hough_geometry*, int32_t, int32_t, int32_t, int32_t,
                                     hough_pipeline**) { return HOUGH_ERR_UNSUPPORTED; }
extern "C" int hough_pipeline_destroy(hough_pipeline*) { return HOUGH_ERR_UNSUPPORTED; }
extern "C" int hough_pipeline_run_host(hough_pipeline*, const float*, int32_t, const int32_t*, int32_t, int32_t, int32_t,
                                       int32_t, int32_t*, int32_t*, hough_candidate*, int32_t, int32_t*, uint8_t*,
                                       int32_t*) { return HOUGH_ERR_UNSUPPORTED; }
