// static_scratch.cu -- the scratch of sa_pack_mask_static: a fixed array in device memory.
//
// Some callers cannot allocate device memory: code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc. sa_pack_mask_static is sa_pack_mask (Sec. 4.1.2,
// M_p = 1(T <= p); K0) with its workspace -- the radix-select histograms, the per-head
// select state and the per-row tie counts -- in the array below instead of a caller's buffer.
// Every GPU that loads the library holds the array (SA_STATIC_SCRATCH_BYTES) until the process
// exits.
//
// In host code the array's NAME is a host-side stand-in, not a device address: a kernel given it
// would fault or, where the GPU can reach host memory, silently use the wrong memory. The address
// comes from cudaGetSymbolAddress, asked once per device with that device current, here in the
// file that defines the array, and is what the kernels receive.
//
// All calls on a device share the array, and it keeps the last call's contents: the pack launcher
// zeroes the histograms on the stream at the start of every call and writes the select state and
// the tie counts before it reads them, so nothing is carried from call to call. Two calls that
// overlap on the GPU (different streams without an ordering between them) race on it.
#include <mutex>

#include "common.cuh"

namespace sa {
namespace {

static __device__ __align__(256) unsigned char g_static_scratch[SA_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_addr[kMaxDevices] = {};

}  // namespace

cudaError_t static_scratch(void** ptr, size_t* bytes) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_mu);
  if (g_addr[dev] == nullptr) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);     // the array's address on the CURRENT device
    if (e != cudaSuccess) return e;
    if (p == nullptr || (reinterpret_cast<uintptr_t>(p) & 255u)) return cudaErrorInvalidSymbol;
    g_addr[dev] = p;
  }
  *ptr = g_addr[dev];
  *bytes = SA_STATIC_SCRATCH_BYTES;
  return cudaSuccess;
}

}  // namespace sa
