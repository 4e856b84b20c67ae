// The PTX wrappers of the tensor-core path live in the public header include/rlxpp_tile.cuh (namespace
// rlxpp_dev::umma), shared by the library's kernels and by rlxpp_dev::TileStream.
#pragma once
#include "../../include/rlxpp_tile.cuh"

namespace rlx {
namespace umma = rlxpp_dev::umma;
}  // namespace rlx
