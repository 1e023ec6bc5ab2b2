// api.cu -- status strings, version and the thread-local CUDA error slot of libxpr.so.
#include "common.cuh"

namespace xpr {
thread_local int32_t g_last_cuda_error = 0;
}

extern "C" const char* xpr_status_string(int32_t status) {
    switch (status) {
        case XPR_OK: return "XPR_OK";
        case XPR_ERR_INVALID_ARG: return "XPR_ERR_INVALID_ARG: null/misaligned pointer, negative size or bad enum";
        case XPR_ERR_CAPACITY: return "XPR_ERR_CAPACITY: more tile-Gaussian pairs than pair_capacity";
        case XPR_ERR_CUDA: return "XPR_ERR_CUDA: CUDA runtime failure (see xpr_last_cuda_error)";
        case XPR_ERR_UNSUPPORTED: return "XPR_ERR_UNSUPPORTED: configuration outside the implemented path";
        default: return "XPR: unknown status";
    }
}

extern "C" int32_t xpr_last_cuda_error(void) { return xpr::g_last_cuda_error; }

extern "C" int32_t xpr_version(void) { return 100; /* 0.1.0 */ }
