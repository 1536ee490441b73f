// torch_shim.cpp -- the only translation unit that sees PyTorch headers.  PyTorch is plumbing
// here: device memory comes from its CUDA caching allocator and work is enqueued on its current
// CUDA stream, so the library cooperates with a host program that also uses torch.
#include <c10/cuda/CUDACachingAllocator.h>
#include <c10/cuda/CUDAStream.h>

#include <cstddef>

extern "C" {

void* lbm_shim_alloc(size_t bytes) {
  try {
    return c10::cuda::CUDACachingAllocator::raw_alloc(bytes);
  } catch (...) {
    return nullptr;
  }
}

void lbm_shim_free(void* p) {
  try {
    if (p) c10::cuda::CUDACachingAllocator::raw_delete(p);
  } catch (...) {
  }
}

// cudaStream_t of torch's current stream on the current device (as void*).
void* lbm_shim_stream(void) {
  try {
    return (void*)c10::cuda::getCurrentCUDAStream().stream();
  } catch (...) {
    return nullptr;
  }
}

}  // extern "C"
