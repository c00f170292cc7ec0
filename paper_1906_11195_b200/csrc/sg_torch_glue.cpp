// sg_torch_glue.cpp -- the only translation unit that includes torch headers.  PyTorch is used
// for exactly two things: device memory (the CUDA caching allocator) and the current stream.
#include <c10/cuda/CUDACachingAllocator.h>
#include <c10/cuda/CUDAFunctions.h>
#include <c10/cuda/CUDAStream.h>

#include <exception>

#include "sg_internal.h"

void *sgx_alloc(size_t bytes)
{
    if (bytes == 0) bytes = 8;
    try {
        if (!c10::cuda::CUDACachingAllocator::get()->initialized()) {
            sg_set_error("torch's CUDA allocator is not initialised: call torch.cuda.init() before sg_create");
            return nullptr;
        }
        return c10::cuda::CUDACachingAllocator::raw_alloc(bytes);
    } catch (const std::exception &e) {
        sg_set_error(std::string("device allocation of ") + std::to_string(bytes) + " bytes failed: " + e.what());
        return nullptr;
    }
}

void sgx_free(void *p)
{
    if (!p) return;
    try {
        c10::cuda::CUDACachingAllocator::raw_delete(p);
    } catch (const std::exception &) {
    }
}

cudaStream_t sgx_stream()
{
    return c10::cuda::getCurrentCUDAStream().stream();
}

int sgx_device_ok(std::string *why)
{
    try {
        if (c10::cuda::device_count() <= 0) {
            if (why) *why = "no CUDA device is visible (this library has no CPU fallback)";
            return 0;
        }
    } catch (const std::exception &e) {
        if (why) *why = e.what();
        return 0;
    }
    return 1;
}
