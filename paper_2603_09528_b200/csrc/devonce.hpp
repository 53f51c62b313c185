// devonce.hpp — per-device, thread-safe one-time configuration for the launch wrappers.
// cudaFuncSetAttribute and occupancy answers belong to ONE device: a process that holds plans on several devices (the
// sharded solve with virtual or real peers) must configure every kernel once per device, and two host threads may
// reach a wrapper at the same time.
#pragma once

#include <cuda_runtime.h>

#include <map>
#include <mutex>
#include <tuple>
#include <utility>

namespace tpt {

class DeviceOnce {
  public:
    // Runs fn() (returning cudaError_t) the first time it is called with a given current device; later calls on that
    // device return cudaSuccess without running it.  A failed fn() is retried on the next call.
    template <class F>
    cudaError_t run(F &&fn) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        std::lock_guard<std::mutex> lock(m_);
        if (dev >= 0 && dev < 64 && (done_ >> dev & 1ull)) return cudaSuccess;
        e = fn();
        if (e == cudaSuccess && dev >= 0 && dev < 64) done_ |= 1ull << dev;
        return e;
    }

  private:
    std::mutex m_;
    unsigned long long done_ = 0;
};

// blocks-per-SM answers of cudaOccupancyMaxActiveBlocksPerMultiprocessor, keyed by (device, threads, dynamic smem)
class OccupancyCache {
  public:
    template <class K>
    cudaError_t get(K kernel, int threads, size_t smem, int *per_sm) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        std::lock_guard<std::mutex> lock(m_);
        const auto key = std::make_tuple(dev, threads, smem);
        auto it = map_.find(key);
        if (it == map_.end()) {
            int v = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, kernel, threads, smem);
            if (e != cudaSuccess) return e;
            it = map_.emplace(key, v).first;
        }
        *per_sm = it->second;
        return cudaSuccess;
    }

  private:
    std::mutex m_;
    std::map<std::tuple<int, int, size_t>, int> map_;
};

// Kernel launch with programmatic dependent launch allowed (ptx.cuh pdl_wait / pdl_launch_dependents): the launch
// latency and prologue of a solve's kernel k+1 overlap the tail of kernel k — what matters on the launch-bound grids.
template <class K, class... Args>
cudaError_t launch_pdl(K kernel, dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args &&...args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

}  // namespace tpt
