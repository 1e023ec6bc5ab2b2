// api.cu -- status strings, version, the thread-local CUDA error slot of libxpr.so, and the loss-gradient helper.
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
        case XPR_ERR_SCRATCH_LIMIT:
            return "XPR_ERR_SCRATCH_LIMIT: these sizes need more workspace than the static scratch of xpr_bin_sort_static "
                   "(XPR_STATIC_SCRATCH_BYTES); use xpr_bin_sort with a caller-provided workspace";
        default: return "XPR: unknown status";
    }
}

extern "C" int32_t xpr_last_cuda_error(void) { return xpr::g_last_cuda_error; }

extern "C" int32_t xpr_version(void) { return 100; /* 0.1.0 */ }

// dL/dimage of the two losses of BASELINE.json's configs (reading C21: sums, not means), one pass over the image:
// kind 0: L = sum |I - target|  ->  sign(I - target);   kind 1: L = sum (I - target)^2  ->  2 (I - target).
namespace xpr {
namespace {
template <int KIND>
__global__ void __launch_bounds__(256) loss_grad_kernel(int64_t n4, int64_t n, const float* __restrict__ image,
                                                        const float* __restrict__ target, float* __restrict__ dL) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    auto g = [](float a, float b) {
        const float d = a - b;
        return KIND == 0 ? (d > 0.0f ? 1.0f : (d < 0.0f ? -1.0f : d)) : 2.0f * d;   // sign(+-0) = +-0, sign(NaN) = NaN
    };
    if (i < n4) {
        const float4 a = reinterpret_cast<const float4*>(image)[i], b = reinterpret_cast<const float4*>(target)[i];
        reinterpret_cast<float4*>(dL)[i] = make_float4(g(a.x, b.x), g(a.y, b.y), g(a.z, b.z), g(a.w, b.w));
    }
    if (i < n - 4 * n4) dL[4 * n4 + i] = g(image[4 * n4 + i], target[4 * n4 + i]);
}
}  // namespace
}  // namespace xpr

extern "C" int32_t xpr_loss_grad(int32_t kind, int64_t n, const float* image, const float* target, float* dL_dimage,
                                 void* stream) {
    using namespace xpr;
    if (kind != 0 && kind != 1) return XPR_ERR_INVALID_ARG;
    if (n < 0) return XPR_ERR_INVALID_ARG;
    if (n == 0) return XPR_OK;
    if (!aligned(image, 16) || !aligned(target, 16) || !aligned(dL_dimage, 16)) return XPR_ERR_INVALID_ARG;
    const int64_t n4 = n / 4;
    const unsigned blocks = (unsigned)((n4 + 255) / 256 + 1);
    if (kind == 0) loss_grad_kernel<0><<<blocks, 256, 0, (cudaStream_t)stream>>>(n4, n, image, target, dL_dimage);
    else           loss_grad_kernel<1><<<blocks, 256, 0, (cudaStream_t)stream>>>(n4, n, image, target, dL_dimage);
    XPR_LAUNCH_CHECK();
    return XPR_OK;
}
