// device_guard.cuh -- every entry point of the C ABI makes its handle's device current for the duration of the
// call and leaves the caller's current device as it found it.
#pragma once
#include <cuda_runtime.h>

namespace pwk {

struct DeviceGuard {
    int prev = -1, dev;
    cudaError_t err;
    explicit DeviceGuard(int d) : dev(d) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        err = (prev == dev) ? cudaSuccess : cudaSetDevice(dev);
    }
    ~DeviceGuard() { if (prev >= 0 && prev != dev) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

}  // namespace pwk
