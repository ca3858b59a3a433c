// Per-device facts and per-(kernel, device) opt-in shared-memory sizes.  Function attributes belong to a device, so
// nothing here is a process-wide flag: a handle created on a second GPU of the same process gets its own entries.
// Thread-safe (planes may be driven from several host threads).
#include <map>
#include <mutex>
#include <utility>

#include "mg_device.h"

namespace mgb {

namespace {
std::mutex g_mu;
std::map<int, DevInfo> g_dev;
std::map<std::pair<const void*, int>, size_t> g_smem;   // (kernel, device) -> bytes configured
}  // namespace

const DevInfo& dev_info() {
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_dev.find(dev);
    if (it != g_dev.end()) return it->second;
    DevInfo d{};
    d.device = dev;
    cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&d.coop, cudaDevAttrCooperativeLaunch, dev);
    if (d.sms <= 0) d.sms = 1;
    return g_dev.emplace(dev, d).first->second;
}

cudaError_t ensure_dyn_smem(const void* func, size_t bytes) {
    int dev = 0;
    cudaGetDevice(&dev);
    std::lock_guard<std::mutex> lk(g_mu);
    auto key = std::make_pair(func, dev);
    auto it = g_smem.find(key);
    if (it != g_smem.end() && it->second >= bytes) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) g_smem[key] = bytes;
    return e;
}

}  // namespace mgb
