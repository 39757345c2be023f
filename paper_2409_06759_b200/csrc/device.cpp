// device.cpp -- per-device facts every launcher needs: the SM count (persistent grids are sized from it) and the
// "first launch of this kernel on this device" test behind the dynamic-shared-memory opt-in.
#include <cuda_runtime.h>

#include <mutex>
#include <set>
#include <utility>

#include "kernels.h"

namespace tcb {

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_mu;
int g_sms[kMaxDevices];
std::set<std::pair<int, const void *>> g_configured;
}  // namespace

int sm_count()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        cudaGetLastError();
        return 148;          // no device (host-only planner): the schedule of a B200
    }
    std::lock_guard<std::mutex> lock(g_mu);
    if (g_sms[dev] == 0) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
            cudaGetLastError();
            n = 148;
        }
        g_sms[dev] = n;
    }
    return g_sms[dev];
}

bool first_use_on_device(const void *tag)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); dev = 0; }
    std::lock_guard<std::mutex> lock(g_mu);
    return g_configured.insert(std::make_pair(dev, tag)).second;
}

}  // namespace tcb
