// common.cuh -- shared host-side helpers of libxpr.so (argument checks, error plumbing).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "xpr.h"

namespace xpr {

extern thread_local int32_t g_last_cuda_error;

inline int32_t cuda_fail(cudaError_t e) {
    g_last_cuda_error = (int32_t)e;
    return XPR_ERR_CUDA;
}

#define XPR_CUDA(call)                                         \
    do {                                                       \
        cudaError_t e__ = (call);                              \
        if (e__ != cudaSuccess) return ::xpr::cuda_fail(e__);  \
    } while (0)

#define XPR_LAUNCH_CHECK() XPR_CUDA(cudaGetLastError())

inline bool aligned(const void* p, size_t a) { return p != nullptr && (reinterpret_cast<uintptr_t>(p) % a) == 0; }

constexpr int TILE = 16;

inline int32_t check_cam_cfg(const xpr_camera* cam, const xpr_config* cfg) {
    if (!cam || !cfg) return XPR_ERR_INVALID_ARG;
    if (cam->width <= 0 || cam->height <= 0) return XPR_ERR_INVALID_ARG;
    if (cam->model != 0 && cam->model != 1) return XPR_ERR_INVALID_ARG;
    if (cfg->projection != 0 && cfg->projection != 1) return XPR_ERR_INVALID_ARG;
    if (cfg->sh_degree < 0) return XPR_ERR_INVALID_ARG;
    if (cfg->sh_degree > 3) return XPR_ERR_UNSUPPORTED;
    if (cfg->tile != TILE) return XPR_ERR_UNSUPPORTED;
    if (cfg->projection == 0 && cam->model != 0) return XPR_ERR_UNSUPPORTED;  // EWA Jacobian is the pinhole's
    if (cfg->views < 0) return XPR_ERR_INVALID_ARG;
    if (cfg->views > XPR_MAX_VIEWS) return XPR_ERR_UNSUPPORTED;
    for (int v = 1; v < cfg->views; ++v)      // a batch of views shares the image geometry (xpr.h)
        if (cam[v].model != cam->model || cam[v].width != cam->width || cam[v].height != cam->height) return XPR_ERR_INVALID_ARG;
    return XPR_OK;
}

inline int num_views(const xpr_config* cfg) { return cfg->views > 1 ? cfg->views : 1; }

inline int tiles_x(const xpr_camera* cam) { return (cam->width + TILE - 1) / TILE; }
inline int tiles_y(const xpr_camera* cam) { return (cam->height + TILE - 1) / TILE; }

}  // namespace xpr
