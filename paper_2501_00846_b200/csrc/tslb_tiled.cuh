// tslb_tiled.cuh -- production kernels: xy-tile + z-marching (placeholder until implemented).
#pragma once
#include "tslb_device.cuh"

namespace tslb {

template <typename T>
int launch_step_tiled(const DevParams<T>& P, const T* S, T* D, cudaStream_t stream,
                      long long* launches, const Marker& mk) {
  (void)mk; (void)P; (void)S; (void)D; (void)stream; (void)launches;
  return int(cudaErrorNotSupported);
}

}  // namespace tslb
