// lm_common.cuh -- small types shared by the kernels of liblm.
#pragma once
#include <stdint.h>

namespace lm {

constexpr int MAX_RHS = 4;   // right-hand sides served by one pair-kernel launch

// Per-right-hand-side pointers (device memory, interleaved xyz, 3N each).
template <typename T> struct RhsIn  { const T* f[MAX_RHS]; const T* t[MAX_RHS]; };   // forces / torques; null = zeros
template <typename T> struct RhsOut { T* lin[MAX_RHS]; T* ang[MAX_RHS]; };           // linear / angular velocities

}  // namespace lm
