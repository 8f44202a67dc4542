// device.cu -- per-device state of the library: SM count and the dynamic shared-memory opt-in of
// the kernels that need more than the 48 KB default. Both are cached per device ordinal under a
// mutex, so a process that uses several GPUs (one after the other or from several threads) gets
// the attribute set on each of them and the right SM count for each.
#include <mutex>

#include "common.cuh"

namespace sa {
namespace {

constexpr int kMaxDevices = 64;
struct DevState {
  int n_sm = 0;
  bool attr[kNumSmemKernels] = {};
};
std::mutex g_mu;
DevState g_dev[kMaxDevices];

}  // namespace

cudaError_t device_sm_count(int* n_sm) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_mu);
  if (g_dev[dev].n_sm == 0) {
    int n = 0;
    e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    g_dev[dev].n_sm = n;
  }
  *n_sm = g_dev[dev].n_sm;
  return cudaSuccess;
}

cudaError_t ensure_dynamic_smem(SmemKernel id, const void* func, int bytes) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_mu);
  if (g_dev[dev].attr[id]) return cudaSuccess;
  e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e != cudaSuccess) return e;
  g_dev[dev].attr[id] = true;
  return cudaSuccess;
}

}  // namespace sa
