// hr_static.cu — hr_dhat_apply_static: the even-odd operator for callers that cannot allocate device memory (code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc).  Dhat is two dependent parity hops with an odd half field between them
// (include/hr_dslash.h, HR_EO_DHAT); every other entry point takes that field from the caller (`tmp`), this one keeps it
// in a file-scope device array of HR_STATIC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.
//
// In host code `hr_static_scratch` is only the handle the runtime registered for the array, not a device address: the address is
// looked up with cudaGetSymbolAddress once per device (that device current) and it is that pointer the kernels get.
#include "hr_common.cuh"

#include <mutex>

static __device__ __align__(256) unsigned char hr_static_scratch[HR_STATIC_SCRATCH_BYTES];

namespace hr {

// Never launched: it names the array in device code, so that the array is kept in the device image whatever the toolchain decides
// about file-scope device variables that only the host refers to.
__global__ void static_scratch_anchor_kernel(unsigned long long* out) {
    if (out) *out = (unsigned long long)(uintptr_t)hr_static_scratch;
}

namespace {
constexpr int MAX_DEVICES = 64;
std::mutex g_scratch_mutex;
void* g_scratch_ptr[MAX_DEVICES];   // device address of hr_static_scratch on device i, nullptr until that device's set-up
}

// Set-up, once per device, with that device current: the device address of the array.
static int static_scratch_address(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        set_error("hr_dhat_apply_static: cudaGetDevice: %s", cudaGetErrorString(e));
        return HR_ECUDA;
    }
    if (dev < 0 || dev >= MAX_DEVICES) {
        set_error("hr_dhat_apply_static: device ordinal %d outside 0..%d", dev, MAX_DEVICES - 1);
        return HR_EUNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, hr_static_scratch);
        if (e != cudaSuccess || !p) {
            set_error("hr_dhat_apply_static: cudaGetSymbolAddress(hr_static_scratch) on device %d: %s", dev,
                      e != cudaSuccess ? cudaGetErrorString(e) : "null address");
            return HR_ECUDA;
        }
        if (reinterpret_cast<uintptr_t>(p) & 255) {
            set_error("hr_dhat_apply_static: the scratch array is not 256-byte aligned on device %d", dev);
            return HR_EALIGN;
        }
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return HR_OK;
}

}  // namespace hr

extern "C" int hr_dhat_apply_static(const hr_geom* g, double m0, const void* u, const void* clover_fwd, const void* clover_inv,
                                    const void* in, void* out, void* stream) {
    using namespace hr;
    if (!geom_ok(g)) {
        set_error("invalid hr_geom (extents must be even and >= 2, volume < 2e9, enums in range)");
        return HR_EINVAL;
    }
    const size_t need = hr_spinor_bytes(g, HR_ODD);
    if (need == 0 || need > (size_t)HR_STATIC_SCRATCH_BYTES) {
        set_error("hr_dhat_apply_static: the odd half field of this lattice takes %zu bytes, the static scratch array holds "
                  "HR_STATIC_SCRATCH_BYTES = %zu; use hr_dirac_eo_apply with a caller-owned tmp",
                  need, (size_t)HR_STATIC_SCRATCH_BYTES);
        return HR_EINVAL;
    }
    void* tmp = nullptr;
    const int rc = static_scratch_address(&tmp);
    if (rc != HR_OK) return rc;
    // Nothing in the array has to start at zero: the first hop writes every entry of the odd half field the second one reads.
    return hr_dirac_eo_apply(g, HR_EO_DHAT, m0, u, clover_fwd, clover_inv, in, out, tmp, stream);
}
