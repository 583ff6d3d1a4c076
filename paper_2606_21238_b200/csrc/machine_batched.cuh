// K3, batched form (placeholder until the warp-cooperative machine lands): forwards to the serial kernel.
#pragma once
#include "machine_serial.cuh"
namespace arc {
inline void launch_machine_batched(const StepParams& P, cudaStream_t s) { arc_machine_serial_kernel<<<1, 32, 0, s>>>(P); }
}  // namespace arc
