// lgs_scan_to_range_image_static: the scan -> range image step (lgs_scan.cu) for callers
// that have no device memory to give as a z-buffer and are not in a position to get any.
//
// Who that is: code that runs where the CUDA allocator must not be touched -- a real-time scan callback whose latency
// budget has no room for a cudaMalloc (it takes a driver lock and may synchronise the whole device), a process whose
// device memory was handed out to a pool at start-up with nothing left over, a plugin inside a host application that
// owns all allocation and gives it none.  Such a caller still has its inputs and outputs (it was given those), but
// the 8 bytes per pixel of z-buffer that lgs_scan_to_range_image asks for are one buffer too many.
//
// So the z-buffer lives here, in the library image: one file-scope __device__ array of LGS_SCAN_STATIC_MAX_PIXELS
// 64-bit words (2 MiB).  The CUDA runtime places it in the global memory of every GPU on which this library's module
// gets loaded and it stays there until the process exits -- that is the price, and the reason the limit is modest.
//
// The name `g_zbuf` means two different things.  In device code it is the array.  In host code it is only a handle
// the runtime uses to look the array up: its host address is NOT where the array lives on the GPU, and a kernel
// handed `g_zbuf` from host code would fault (or scribble over host memory on a system where the GPU can reach it).
// The device address comes from cudaGetSymbolAddress, asked for once per device with that device current, in this
// translation unit (the symbol is static: no other file can name it), and that address is what the kernels get.
#include <mutex>

#include "lgs_internal.cuh"

namespace lgs {
namespace {

static __device__ __align__(256) unsigned long long g_zbuf[LGS_SCAN_STATIC_MAX_PIXELS];

constexpr int kMaxDevices = 64;        // device ordinals with a cached address; higher ordinals look it up every call
std::mutex g_mu;
void* g_zbuf_addr[kMaxDevices] = {nullptr};

// Device address of g_zbuf on the CURRENT device.  The first call on a device asks the runtime (which loads the module
// there if it is not loaded yet -- not something to do inside a stream capture); later calls read the cache.
cudaError_t zbuf_address(void** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const bool cached = dev >= 0 && dev < kMaxDevices;
  std::lock_guard<std::mutex> lock(g_mu);
  if (cached && g_zbuf_addr[dev]) { *out = g_zbuf_addr[dev]; return cudaSuccess; }
  void* p = nullptr;
  e = cudaGetSymbolAddress(&p, g_zbuf);
  if (e != cudaSuccess) return e;
  if (!p) return cudaErrorInvalidSymbol;
  if (cached) g_zbuf_addr[dev] = p;
  *out = p;
  return cudaSuccess;
}

}  // namespace
}  // namespace lgs

extern "C" lgs_status lgs_scan_to_range_image_static(const float* points, const float* normals, int64_t M,
                                                     const lgs_sensor* s, float* out_range, float* out_normal,
                                                     lgs_stream stream) {
  if (!s || s->H < 1 || s->W < 1) return LGS_ERR_INVALID_ARG;
  if ((int64_t)s->H * (int64_t)s->W > (int64_t)LGS_SCAN_STATIC_MAX_PIXELS) return LGS_ERR_STATIC_LIMIT;
  void* zbuf = nullptr;
  if (lgs::zbuf_address(&zbuf) != cudaSuccess) return LGS_ERR_CUDA;
  // From here on this is the ordinary call, pointed at the built-in z-buffer: same argument checks, same three kernels
  // (the first of which resets every word the image uses, so what the previous call left behind does not matter).
  return lgs_scan_to_range_image(points, normals, M, s, zbuf, sizeof(unsigned long long) * LGS_SCAN_STATIC_MAX_PIXELS,
                                 out_range, out_normal, stream);
}
